"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances (BASELINE.json north_star): relative L2 error per
operator application <= 1e-12 in fp64 and <= 2e-6 in fp32 (the fp32 path receives the fp64 inputs rounded
to nearest; the oracle keeps the fp64 originals).  Solves: true residual <= 1e-10 (1.05e-10 with drift),
iteration counts within max(1, ceil(2 %)) of the oracle's.
"""
import json
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL = {torch.float64: 1e-12, torch.float32: 2e-6}
GOLD = os.path.join(os.path.dirname(__file__), "golden", "solver_golden.json")


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def cola_mod():
    from paper_2302_00850_b200 import binding

    assert torch.cuda.is_available()
    return binding


class Case:
    """Links + oracle-side fields for one lattice, and a CUDA context per link format."""

    def __init__(self, binding, dims, kind, kappa, csw, bc=BC, seed=5, eps=0.3):
        self.dims, self.kappa, self.csw, self.bc = dims, kappa, csw, bc
        if kind == "haar":
            self.U = inputs.links_haar(dims, seed)
        elif kind == "unit":
            self.U = inputs.links_unit(dims)
        else:
            self.U = inputs.links_smooth(dims, eps, seed)
        self.Un = self.U.numpy()
        self.A = oracle.clover(dims, self.Un, kappa, csw)
        self.Ainv = oracle.clover_inverse(self.A)
        self.binding = binding
        self._ctx = {}
        self.par = oracle.parity_mask(dims)

    def ctx(self, compress12=True):
        if compress12 not in self._ctx:
            c = self.binding.Cola(self.dims, self.kappa, self.csw, bc=self.bc, compress12=compress12)
            c.gauge_upload(self.U)
            self._ctx[compress12] = c
        return self._ctx[compress12]

    def spinor(self, seed):
        return inputs.source_gaussian(self.dims, seed)

    def mask(self, p):
        return (self.par == p)[..., None, None]


CASES = {
    "2^4 haar": dict(dims=(2, 2, 2, 2), kind="haar", kappa=0.12, csw=1.0),
    "4^4 haar (config 0)": dict(dims=(4, 4, 4, 4), kind="haar", kappa=0.12, csw=1.0, seed=inputs.config_seed_links(0)),
    "4x2x6x2 smooth": dict(dims=(4, 2, 6, 2), kind="smooth", kappa=0.124, csw=1.3),
    "6x4x2x8 all-antiperiodic": dict(dims=(6, 4, 2, 8), kind="smooth", kappa=0.12, csw=0.7, bc=(-1, -1, -1, -1)),
    "12x10x6x4 ragged tail": dict(dims=(12, 10, 6, 4), kind="smooth", kappa=0.1245, csw=1.0),
    "8^3x16 smooth": dict(dims=(8, 8, 8, 16), kind="smooth", kappa=0.1245, csw=1.0),
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request, cola_mod):
    return Case(cola_mod, **CASES[request.param])


def to_dev(t, dtype):
    ct = torch.complex128 if dtype == torch.float64 else torch.complex64
    return t.to(ct).cuda()


# ---------------------------------------------------------------------------------------------
# T2: layout round trips
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_pack_unpack_roundtrip_and_layout(case, dtype):
    c = case.ctx()
    psi = to_dev(case.spinor(3), dtype)
    internal = c.spinor_pack(psi)
    assert torch.equal(c.spinor_unpack(internal), psi)
    # the documented layout: [parity][chunk][Vh][reals], cb = (x>>1) + Xh*(y + Y*(z + Z*t))
    lx, ly, lz, lt = case.dims
    n = internal.shape[-1]
    host = internal.cpu().numpy()
    ref = torch.view_as_real(psi.cpu()).numpy().reshape(lt, lz, ly, lx, 24)
    rng = np.random.default_rng(0)
    for _ in range(50):
        x, y, z, t = (int(rng.integers(0, d)) for d in case.dims)
        p = (x + y + z + t) & 1
        cb = (x >> 1) + (lx // 2) * (y + ly * (z + lz * t))
        got = host[p, :, cb, :].reshape(24)
        assert np.array_equal(got, ref[t, z, y, x]), (x, y, z, t, n)


def test_precision_convert_roundtrip(case):
    c = case.ctx()
    psi = to_dev(case.spinor(4), torch.float64)
    i64 = c.spinor_pack(psi)
    i32 = c.spinor_convert(i64, torch.float32)
    assert torch.equal(c.spinor_unpack(i32), psi.to(torch.complex64))
    back = c.spinor_convert(i32, torch.float64)
    assert torch.equal(c.spinor_unpack(back), psi.to(torch.complex64).to(torch.complex128))
    half = c.spinor_convert(i64[1].contiguous(), torch.float32)
    assert torch.equal(half, i32[1])


# ---------------------------------------------------------------------------------------------
# H1/H2: clover field and its inverse
# ---------------------------------------------------------------------------------------------
def test_clover_build_and_inverse_match_oracle(case):
    c = case.ctx()
    A = c.clover_unpack(0).cpu().numpy()
    assert rel(A, case.A) < 1e-13
    Ainv = c.clover_unpack(1).cpu().numpy()
    odd = case.par == 1
    assert rel(Ainv[odd], case.Ainv[odd]) < 1e-12
    assert np.abs(Ainv[~odd]).max() == 0
    assert c.gauge_info() < 1e-13


# ---------------------------------------------------------------------------------------------
# T3: operators
# ---------------------------------------------------------------------------------------------
FORMATS = [(torch.float64, True), (torch.float32, True), (torch.float32, False)]


@pytest.mark.parametrize("dtype,compress12", FORMATS)
@pytest.mark.parametrize("parity", [0, 1])
def test_parity_dslash(case, dtype, compress12, parity):
    c = case.ctx(compress12)
    psi = case.spinor(11)
    want = oracle.dslash_parity(case.dims, case.bc, case.Un, parity, psi.numpy())
    internal = c.spinor_pack(to_dev(psi, dtype))
    out = torch.zeros_like(internal)
    c.dslash_apply(parity, internal[1 - parity].contiguous(), out=out[parity])
    got = c.spinor_unpack(out).cpu().numpy()
    assert rel(got, want) < TOL[dtype]
    assert np.abs(got[case.par != parity]).max() == 0


@pytest.mark.parametrize("dtype,compress12", FORMATS)
@pytest.mark.parametrize("dagger", [False, True])
def test_fermion_matrix(case, dtype, compress12, dagger):
    c = case.ctx(compress12)
    psi = case.spinor(12)
    want = oracle.M(case.dims, case.bc, case.Un, case.A, case.kappa, psi.numpy(), dagger=dagger)
    got = c.spinor_unpack(c.fermion_matrix_apply(c.spinor_pack(to_dev(psi, dtype)), dagger=dagger)).cpu().numpy()
    assert rel(got, want) < TOL[dtype]


@pytest.mark.parametrize("dtype,compress12", FORMATS)
@pytest.mark.parametrize("dagger", [False, True])
def test_schur_operator(case, dtype, compress12, dagger):
    c = case.ctx(compress12)
    psi = case.spinor(13) * case.mask(0)
    want = oracle.schur(case.dims, case.bc, case.Un, case.A, case.Ainv, case.kappa, psi.numpy(), dagger=dagger)
    internal = c.spinor_pack(to_dev(psi, dtype))
    out = torch.zeros_like(internal)
    c.schur_apply(internal[0].contiguous(), dagger=dagger, out=out[0])
    got = c.spinor_unpack(out).cpu().numpy()
    assert rel(got, want) < TOL[dtype]


def test_host_entry_points_match_device_entry_points(case):
    c = case.ctx()
    psi = case.spinor(14)
    want = oracle.M(case.dims, case.bc, case.Un, case.A, case.kappa, psi.numpy())
    got = c.fermion_matrix_apply_host(psi.pin_memory())
    assert rel(got.numpy(), want) < 1e-12
    got32 = c.fermion_matrix_apply_host(psi.to(torch.complex64).pin_memory())
    assert rel(got32.numpy(), want) < 2e-6
    wantd = oracle.dslash_parity(case.dims, case.bc, case.Un, 1, psi.numpy())
    gotd = c.dslash_apply_host(1, psi.pin_memory())
    assert rel(gotd.numpy(), wantd) < 1e-12


# ---------------------------------------------------------------------------------------------
# T4: solvers
# ---------------------------------------------------------------------------------------------
def iter_ok(n_gpu, n_ref):
    return abs(n_gpu - n_ref) <= max(1, math.ceil(0.02 * n_ref))


@pytest.mark.parametrize("even_odd", [False, True])
@pytest.mark.parametrize("mixed", [False, True])
def test_cg_solve_small(case, even_odd, mixed):
    if case.dims == (8, 8, 8, 16) and not even_odd:
        pytest.skip("unpreconditioned CGNR at 8^3x16 is covered by the even-odd case")
    c = case.ctx()
    b = case.spinor(21)
    ref = oracle.cgnr(case.dims, case.bc, case.Un, case.A, case.Ainv, case.kappa, b.numpy(), even_odd=even_odd, tol=1e-10)
    assert ref["converged"]
    x, info = c.cg_solve(b.cuda(), tol=1e-10, even_odd=even_odd, mixed=mixed)
    assert info["converged"]
    assert info["true_residual"] <= 1.05e-10
    # recompute the true residual with the ORACLE's operator
    xn = x.cpu().numpy()
    res = np.linalg.norm((b.numpy() - oracle.M(case.dims, case.bc, case.Un, case.A, case.kappa, xn)).ravel()) / np.linalg.norm(b.numpy().ravel())
    assert res <= 1.05e-10
    assert abs(res - info["true_residual"]) <= 1e-3 * res + 1e-14
    assert iter_ok(info["iters"], ref["iters"]), (info["iters"], ref["iters"])
    assert rel(xn, ref["x"]) < 5e-9
    if mixed:
        assert info["reliable_updates"] >= 1
    # host-buffer entry point gives the same answer
    if even_odd or not mixed:
        xh, infoh = c.cg_solve(b.pin_memory(), tol=1e-10, even_odd=even_odd, mixed=mixed)
        assert infoh["iters"] == info["iters"]
        assert rel(xh.numpy(), xn) < 1e-12


def test_cg_dense_inverse_on_2to4(cola_mod):
    import bruteforce as bf

    case = Case(cola_mod, (2, 2, 2, 2), "haar", 0.12, 1.0, seed=51)
    Md = bf.dense_M(case.dims, BC, case.Un, 0.12, 1.0)
    b = case.spinor(52)
    x_exact = np.linalg.solve(Md, b.numpy().ravel())
    for eo in (False, True):
        x, info = case.ctx().cg_solve(b.cuda(), even_odd=eo)
        assert info["converged"] and rel(x.cpu().numpy().ravel(), x_exact) < 5e-9


def test_config0_and_config1_against_stored_oracle_results(cola_mod):
    """BASELINE.json configs 0 and 1 at full size; expected values written by tests/golden/make_golden.py (oracle only)."""
    gold = json.load(open(GOLD))
    for k, modes in ((0, ("full", "eo")), (1, ("eo",))):
        cfg = inputs.CONFIGS[k]
        U = inputs.make_links(k)
        b = inputs.make_source(k, u=U)
        c = cola_mod.Cola(cfg["dims"], cfg["kappa"], cfg["csw"], compress12=True)
        c.gauge_upload(U)
        for mode in modes:
            g = gold[str(k)][mode]
            for mixed in (False, True):
                x, info = c.cg_solve(b.cuda(), even_odd=(mode == "eo"), mixed=mixed)
                assert info["converged"] and info["true_residual"] <= 1.05e-10
                assert iter_ok(info["iters"], g["iters"]), (k, mode, mixed, info["iters"], g["iters"])
                xs = x.cpu().numpy().reshape(-1, 12)[np.array(g["sites"])]
                want = np.array(g["x_re"]) + 1j * np.array(g["x_im"])
                assert np.linalg.norm(xs - want) / np.linalg.norm(want) < 5e-8
                assert abs(np.linalg.norm(x.cpu().numpy().ravel()) - g["x_norm"]) / g["x_norm"] < 1e-8
        c.close()


def test_config1_schur_applied_100_times(cola_mod):
    """BJ:c1: even-odd operator applied 100x (ping-pong); compare with the oracle after 3 and check the
    100-fold product stays finite and deterministic."""
    cfg = inputs.CONFIGS[1]
    U = inputs.make_links(1)
    Un = U.numpy()
    A = oracle.clover(cfg["dims"], Un, cfg["kappa"], cfg["csw"])
    Ainv = oracle.clover_inverse(A)
    c = cola_mod.Cola(cfg["dims"], cfg["kappa"], cfg["csw"])
    c.gauge_upload(U)
    par = oracle.parity_mask(cfg["dims"])
    psi = inputs.make_source(1, u=U) * torch.from_numpy((par == 0)[..., None, None])
    want = psi.numpy()
    for _ in range(3):
        want = oracle.schur(cfg["dims"], BC, Un, A, Ainv, cfg["kappa"], want)
    for dtype in (torch.float64, torch.float32):
        internal = c.spinor_pack(to_dev(psi, dtype))
        runs = []
        for rep in range(2):
            a, b_ = internal[0].clone(), torch.empty_like(internal[0])
            for n in range(1, 101):
                c.schur_apply(a, out=b_)
                a, b_ = b_, a
                if n == 3 and rep == 0:
                    full = torch.zeros_like(internal)
                    full[0] = a
                    assert rel(c.spinor_unpack(full).cpu().numpy(), want) < 3 * TOL[dtype]
            runs.append(a.clone())
        assert torch.equal(runs[0], runs[1])           # deterministic
        if dtype == torch.float64:
            assert torch.isfinite(runs[0]).all()
    c.close()


# ---------------------------------------------------------------------------------------------
# error behaviour of the ABI
# ---------------------------------------------------------------------------------------------
def test_error_codes(cola_mod):
    b = cola_mod
    with pytest.raises(b.ColaError) as e:
        b.Cola((3, 4, 4, 4), 0.12, 1.0)
    assert e.value.status == b.COLA_EINVAL
    c = b.Cola((4, 4, 4, 4), 0.12, 1.0)
    x = torch.zeros(6, c.Vh, 4, device="cuda")
    with pytest.raises(b.ColaError) as e:
        c.dslash_apply(0, x)
    assert e.value.status == b.COLA_ENOTREADY
    with pytest.raises(b.ColaError) as e:
        c.set_workspace(torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.status == b.COLA_ENOMEM
    # non-unitary links are rejected when 12-real compression is on, accepted otherwise
    U = inputs.links_haar((4, 4, 4, 4), 1)
    bad = U.clone()
    bad[0, 0, 0, 0, 0] *= 1.001
    with pytest.raises(b.ColaError) as e:
        c.gauge_upload(bad)
    assert e.value.status == b.COLA_EINVAL
    c18 = b.Cola((4, 4, 4, 4), 0.12, 1.0, compress12=False)
    c18.gauge_upload(bad)
    assert c18.gauge_info() > 1e-4
    # max_iter -> COLA_ENOCONV with info filled and the last iterate returned
    c.gauge_upload(U)
    src = inputs.source_gaussian((4, 4, 4, 4), 2).cuda()
    xx, info = c.cg_solve(src, max_iter=3)
    assert not info["converged"] and info["iters"] == 3 and 0 < info["true_residual"] < 1
    with pytest.raises(b.ColaError) as e:
        c.cg_solve(src, tol=-1.0)
    assert e.value.status == b.COLA_EINVAL
    bad_src = src.clone()
    bad_src[1, 2, 3, 0, 1, 1] = float("nan")
    for kw in (dict(mixed=0), dict(mixed=1)):
        with pytest.raises(b.ColaError) as e:
            c.cg_solve(bad_src, **kw)
        assert e.value.status == b.COLA_EINVAL and "NaN" in str(e.value)
    with pytest.raises(b.ColaError) as e:
        c.cg_solve_mrhs(torch.stack([src, bad_src]))
    assert e.value.status == b.COLA_EINVAL
    xx, info = c.cg_solve(src)                       # the context is still usable afterwards
    assert info["converged"]


def test_device_links_upload_equals_host_upload(cola_mod):
    dims = (4, 4, 4, 8)
    U = inputs.links_smooth(dims, 0.3, 9)
    a = cola_mod.Cola(dims, 0.1245, 1.0)
    a.gauge_upload(U)
    d = cola_mod.Cola(dims, 0.1245, 1.0)
    d.gauge_upload(U.cuda())
    psi = inputs.source_gaussian(dims, 3).to(torch.complex64).cuda()
    ya = a.fermion_matrix_apply(a.spinor_pack(psi))
    yd = d.fermion_matrix_apply(d.spinor_pack(psi))
    assert torch.equal(ya, yd)


def test_profile_kernel_counts_the_dominant_kernel_only(cola_mod):
    dims = (8, 8, 8, 16)
    c = cola_mod.Cola(dims, 0.1245, 1.0)
    c.gauge_upload(inputs.links_smooth(dims, 0.3, 9))
    v32 = c.spinor_pack(inputs.source_gaussian(dims, 3).to(torch.complex64).cuda())
    v64 = c.spinor_pack(inputs.source_gaussian(dims, 3).cuda())
    assert c.profile_result() == (0.0, 0, 0)
    c.profile_kernel(True)
    for _ in range(5):
        c.schur_apply(v32[0].contiguous())          # one fused dslash+clover+xpay launch each (kernel 2)
    c.fermion_matrix_apply(v32)                      # two
    c.schur_apply(v64[0].contiguous())               # fp64: not the inner-precision kernel, not counted
    c.dslash_apply(0, v32[1].contiguous())           # plain dslash: not counted
    ms, n, skipped = c.profile_result()
    assert n == 7 and skipped == 0 and 0 < ms < 5
    # a mixed solve: 2 per iteration + the start-up application, speculative no-ops reported apart
    x, info = c.cg_solve(inputs.source_gaussian(dims, 4).cuda(), mixed=1)
    ms, n, skipped = c.profile_result()
    # (on a lattice this small a working launch is not much longer than a no-op, so only the total is exact)
    assert 2 * info["iters"] + 1 <= n + skipped <= 2 * info["iters"] + 1 + 2 * info["reliable_updates"] and n > info["iters"]
    c.profile_kernel(False)
    c.schur_apply(v32[0].contiguous())
    assert c.profile_result() == (0.0, 0, 0)
    c.close()


def test_everything_runs_on_the_callers_stream(cola_mod):
    """The context launches on the stream it was given (torch's current stream at creation, or cola_set_stream): a solve
    on a side stream, with the inputs produced on that stream right before, gives the default-stream result bit for bit."""
    dims = (8, 8, 8, 16)
    U = inputs.links_smooth(dims, 0.3, 9)
    b_host = inputs.source_gaussian(dims, 5)
    c0 = cola_mod.Cola(dims, 0.1245, 1.0)
    c0.gauge_upload(U)
    x0, info0 = c0.cg_solve(b_host.cuda(), mixed=1)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        c1 = cola_mod.Cola(dims, 0.1245, 1.0)          # picks up `side`
        c1.gauge_upload(U)
        b = b_host.cuda(non_blocking=True) * 1.0        # produced on `side` just before the solve
        x1, info1 = c1.cg_solve(b, mixed=1)
        v = c1.spinor_pack(b.to(torch.complex64))
        y1 = c1.schur_apply(v[0].contiguous())
    side.synchronize()
    assert info1["iters"] == info0["iters"] and torch.equal(x1, x0)
    y0 = c0.schur_apply(c0.spinor_pack(b_host.to(torch.complex64).cuda())[0].contiguous())
    torch.cuda.synchronize()
    assert torch.equal(y0, y1)
    # cola_set_stream moves an existing context
    c0.set_stream(side.cuda_stream)
    with torch.cuda.stream(side):
        x2, info2 = c0.cg_solve(b_host.cuda(), mixed=1)
    side.synchronize()
    assert torch.equal(x2, x0)
    c0.close()
    c1.close()
