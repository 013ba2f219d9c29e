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


EPS = {torch.float64: 2.0 ** -52, torch.float32: 2.0 ** -23}


def check_op(got, want, dtype):
    """north_star's tolerance on the relative L2 error, and beside it a bound on every single real component: on a
    large lattice one component wrong by a per cent moves the L2 norm by less than the fp32 tolerance, so the norm
    alone would not see it.  An output component is a sum of ~100 products of magnitude <= max|psi|; its rounding
    error (inputs rounded to the working precision included) is a few eps * sqrt(100) * rms, far below
    64 eps * max|want|, while a dropped or mis-signed term is of order rms ~ 0.1 max|want|."""
    assert rel(got, want) < TOL[dtype]
    assert np.abs(np.asarray(got) - np.asarray(want)).max() <= 64 * EPS[dtype] * np.abs(want).max()


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
    check_op(got, want, dtype)
    assert np.abs(got[case.par != parity]).max() == 0


@pytest.mark.parametrize("dtype,compress12", FORMATS)
@pytest.mark.parametrize("dagger", [False, True])
def test_fermion_matrix(case, dtype, compress12, dagger):
    c = case.ctx(compress12)
    psi = case.spinor(12)
    want = oracle.M(case.dims, case.bc, case.Un, case.A, case.kappa, psi.numpy(), dagger=dagger)
    got = c.spinor_unpack(c.fermion_matrix_apply(c.spinor_pack(to_dev(psi, dtype)), dagger=dagger)).cpu().numpy()
    check_op(got, want, dtype)


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
    check_op(got, want, dtype)


def test_host_entry_points_match_device_entry_points(case):
    c = case.ctx()
    psi = case.spinor(14)
    want = oracle.M(case.dims, case.bc, case.Un, case.A, case.kappa, psi.numpy())
    got = c.fermion_matrix_apply_host(psi.pin_memory())
    check_op(got.numpy(), want, torch.float64)
    got32 = c.fermion_matrix_apply_host(psi.to(torch.complex64).pin_memory())
    check_op(got32.numpy(), want, torch.float32)
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
        # SURVEY O8's reliable-update schedule: the passes after which the fp64 residual is recomputed follow from the
        # ORACLE's fp64 residual history alone (tests/schedule.py; pinned against oracle.cgnr_mixed on the CPU)
        from schedule import reliable_update_schedule

        rhs = oracle.eo_prepare(case.dims, case.bc, case.Un, case.Ainv, case.kappa, b.numpy()) if even_odd else b.numpy()
        rmax0 = np.linalg.norm(rhs.ravel()) / np.linalg.norm(b.numpy().ravel())
        want_upd, margin = reliable_update_schedule(ref["history"], rmax0, 0.1, 1e-10)
        xh_, ih = c.cg_solve_history(b.cuda(), tol=1e-10, even_odd=even_odd, mixed=mixed)
        assert ih["iters"] == info["iters"] and ih["reliable_updates"] == info["reliable_updates"] and torch.equal(xh_, x)
        assert len(ih["update_iters"]) == info["reliable_updates"]
        own, own_margin = reliable_update_schedule(ih["history"], rmax0, 0.1, 1e-10)
        if own_margin > 1e-5:
            assert ih["update_iters"] == own, (ih["update_iters"], own)     # the rule on the solver's own recurrence
        if even_odd and margin > 1e-3:
            assert ih["update_iters"] == want_upd, (ih["update_iters"], want_upd)
        else:   # unpreconditioned M: the fp32 recurrence lags the fp64 one by less than a pass (test_oracle_pins.py)
            assert abs(info["reliable_updates"] - len(want_upd)) <= 1
            assert all(min(abs(u - w) for w in want_upd) <= 1 for u in ih["update_iters"]), (ih["update_iters"], want_upd)
    # host-buffer entry point gives the same answer
    xh, infoh = c.cg_solve(b.pin_memory(), tol=1e-10, even_odd=even_odd, mixed=mixed)
    assert infoh["iters"] == info["iters"] and infoh["reliable_updates"] == info["reliable_updates"]
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
    # ... but their 16-bit copy (always 12 reals + rebuilt third row) would be wrong: the H16 operator and mixed = 2 refuse
    v18 = c18.spinor_pack(inputs.source_gaussian((4, 4, 4, 4), 2).to(torch.complex64).cuda())
    c18.fermion_matrix_apply(v18)                                   # fp32 x18: fine
    with pytest.raises(b.ColaError) as e:
        c18.fermion_matrix_apply(v18, h16=True)
    assert e.value.status == b.COLA_EINVAL and "16-bit" in str(e.value)
    for solve in (lambda: c18.cg_solve(inputs.source_gaussian((4, 4, 4, 4), 2).cuda(), mixed=2),
                  lambda: c18.cg_solve_mrhs(torch.stack([inputs.source_gaussian((4, 4, 4, 4), 2).cuda()] * 2), mixed=2)):
        with pytest.raises(b.ColaError) as e:
            solve()
        assert e.value.status == b.COLA_EINVAL
    xx18, info18 = c18.cg_solve(inputs.source_gaussian((4, 4, 4, 4), 2).cuda(), mixed=1)
    assert info18["converged"]
    c18.close()
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
    # spinor layout calls take COLA_F64 / COLA_F32 only (COLA_F32_H16 is an operator precision, not a spinor format)
    import ctypes
    lib = ctypes.CDLL(b.lib_path())
    v64 = c.spinor_pack(src)
    dst = torch.empty_like(v64)
    for call in (lambda: lib.cola_spinor_convert(c._h, b.COLA_F32_H16, ctypes.c_void_p(v64.data_ptr()), ctypes.c_void_p(dst.data_ptr()), 2),
                 lambda: lib.cola_spinor_pack(c._h, b.COLA_F32_H16, ctypes.c_void_p(src.data_ptr()), ctypes.c_void_p(dst.data_ptr())),
                 lambda: lib.cola_spinor_unpack(c._h, 7, ctypes.c_void_p(v64.data_ptr()), ctypes.c_void_p(dst.data_ptr()))):
        assert call() == b.COLA_EINVAL
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


def test_nan_links_stop_the_solvers_instead_of_iterating_to_max_iter(cola_mod):
    """A NaN that enters through the gauge field (not the source) never satisfies a stopping test: the solvers must
    notice the non-finite residual and return COLA_EINVAL (single and batched), not run to max_iter."""
    b = cola_mod
    dims = (4, 4, 4, 4)
    U = inputs.links_haar(dims, 1)
    bad = U.clone()
    bad[1, 2, 3, 0, 2, 1, 1] = float("nan")
    c = b.Cola(dims, 0.12, 1.0, compress12=False)      # compress12 would reject the link (NaN is "not unitary")
    try:
        c.gauge_upload(bad)
    except b.ColaError as ex:                          # NaN pivot in the clover inverse: also a clean refusal
        assert ex.status == b.COLA_EINVAL
        return
    src = inputs.source_gaussian(dims, 2).cuda()
    for solve in (lambda: c.cg_solve(src, mixed=1, max_iter=200), lambda: c.cg_solve(src, mixed=0, max_iter=200),
                  lambda: c.cg_solve_mrhs(torch.stack([src, src]), max_iter=200)):
        with pytest.raises(b.ColaError) as e:
            solve()
        assert e.value.status == b.COLA_EINVAL
    c.close()


def test_features_select_the_carved_fields(cola_mod):
    """cola_set_features: without COLA_FEAT_FULL_M / COLA_FEAT_H16 the workspace is smaller, everything the even-odd
    mixed solver needs still works and gives the same bits, and calls that need a missing field return COLA_EINVAL."""
    b = cola_mod
    dims = (8, 8, 8, 16)
    U = inputs.links_smooth(dims, 0.3, 9)
    src = inputs.source_gaussian(dims, 5).cuda()
    full = b.Cola(dims, 0.1245, 1.0)
    lean = b.Cola(dims, 0.1245, 1.0, features=0)
    assert lean.workspace_bytes() < 0.86 * full.workspace_bytes()
    full.gauge_upload(U)
    lean.gauge_upload(U)
    x0, i0 = full.cg_solve(src, mixed=1)
    x1, i1 = lean.cg_solve(src, mixed=1)
    assert torch.equal(x0, x1) and i0["iters"] == i1["iters"]
    xh, ih = lean.cg_solve(src.cpu().pin_memory(), mixed=1)
    assert torch.equal(xh.cuda(), x1)
    v32 = lean.spinor_pack(src.to(torch.complex64))
    v64 = lean.spinor_pack(src)
    assert torch.equal(lean.schur_apply(v32[0].contiguous()), full.schur_apply(v32[0].contiguous()))
    assert torch.equal(lean.dslash_apply(1, v32[0].contiguous()), full.dslash_apply(1, v32[0].contiguous()))
    assert torch.equal(lean.fermion_matrix_apply(v64), full.fermion_matrix_apply(v64))      # fp64 M is always there
    for call in (lambda: lean.fermion_matrix_apply(v32), lambda: lean.schur_apply(v32[0].contiguous(), h16=True),
                 lambda: lean.cg_solve(src, mixed=2), lambda: lean.cg_solve(src, even_odd=False),
                 lambda: lean.fermion_matrix_apply_mrhs(torch.stack([v32, v32]))):
        with pytest.raises(b.ColaError) as e:
            call()
        assert e.value.status == b.COLA_EINVAL
    assert torch.equal(lean.schur_apply_mrhs(torch.stack([v32[0], v32[0]]))[1], full.schur_apply(v32[0].contiguous()))
    # operators-only multi-rhs workspace: smaller, and the batched solver says it needs the large one
    assert lean.mrhs_workspace_bytes(4, for_solver=False) < 0.3 * lean.mrhs_workspace_bytes(4, for_solver=True)
    lean.set_mrhs_workspace(2, for_solver=False)
    import ctypes
    sp = lean._solve_params(1e-10, 100, True, 1, 0.1)
    infos = (b.ColaSolveInfo * 2)()
    bs = torch.stack([src, src])
    xs = torch.empty_like(bs)
    st = ctypes.CDLL(b.lib_path()).cola_cg_solve_mrhs(lean._h, ctypes.byref(sp), 2, ctypes.c_void_p(bs.data_ptr()), ctypes.c_void_p(xs.data_ptr()), infos)
    assert st == b.COLA_ENOTREADY
    xs, infos = lean.cg_solve_mrhs(bs)        # the binding re-lends a solver-sized workspace
    assert torch.equal(xs[0], x1) and torch.equal(xs[1], x1)
    # H16 alone
    h = b.Cola(dims, 0.1245, 1.0, features=b.COLA_FEAT_H16)
    h.gauge_upload(U)
    x2, i2 = h.cg_solve(src, mixed=2)
    x3, i3 = full.cg_solve(src, mixed=2)
    assert torch.equal(x2, x3)
    for c in (full, lean, h):
        c.close()


def test_smallest_pivot_is_reported_and_indefinite_blocks_are_refused(cola_mod):
    """the upload reports the smallest pivot of the 6x6 inversions; a block that is not positive definite
    (here: csw pushed far beyond anything physical on rough links) is COLA_EINVAL, not a silent garbage inverse."""
    b = cola_mod
    dims = (4, 4, 4, 4)
    U = inputs.links_haar(dims, 3)
    Un = U.numpy()
    c = b.Cola(dims, 0.12, 1.0)
    c.gauge_upload(U)
    A = oracle.clover(dims, Un, 0.12, 1.0)
    odd = oracle.parity_mask(dims) == 1
    ev = np.linalg.eigvalsh(np.concatenate([A[odd][:, :6, :6], A[odd][:, 6:, 6:]]))
    piv = c.clover_info()
    # an unpivoted elimination of a Hermitian positive-definite block has pivots between its extreme eigenvalues
    assert ev.min() - 1e-12 <= piv <= ev.max() and piv > 0
    # brute force: the same elimination in numpy on the oracle's blocks
    blocks = np.concatenate([A[odd][:, :6, :6], A[odd][:, 6:, 6:]])
    pmin = np.inf
    for blk in blocks:
        m = blk.copy()
        for k in range(6):
            pmin = min(pmin, m[k, k].real)
            m[k + 1:, :] -= np.outer(m[k + 1:, k] / m[k, k], m[k, :])
    assert abs(piv - pmin) <= 1e-12
    c.close()
    csw_bad = 40.0
    Abad = oracle.clover(dims, Un, 0.12, csw_bad)
    assert np.linalg.eigvalsh(np.concatenate([Abad[odd][:, :6, :6], Abad[odd][:, 6:, 6:]])).min() < 0
    cb = b.Cola(dims, 0.12, csw_bad)
    with pytest.raises(b.ColaError) as e:
        cb.gauge_upload(U)
    assert e.value.status == b.COLA_EINVAL and "positive definite" in str(e.value)
    assert cb.clover_info() <= 0
    with pytest.raises(b.ColaError) as e:
        cb.dslash_apply(0, torch.zeros(6, cb.Vh, 4, device="cuda"))
    assert e.value.status == b.COLA_ENOTREADY
    cb.close()


def test_a_missing_device_surfaces_as_COLA_ECUDA(cola_mod):
    """COLA_ECUDA (SURVEY 8(b) error cases): a device ordinal that does not exist."""
    b = cola_mod
    import ctypes
    lib = ctypes.CDLL(b.lib_path())
    lib.cola_last_error.restype = ctypes.c_char_p
    lib.cola_last_error.argtypes = [ctypes.c_void_p]
    p = b.ColaParams()
    p.dims[:] = (4, 4, 4, 4)
    p.bc[:] = (1, 1, 1, -1)
    p.kappa, p.csw, p.device = 0.12, 1.0, torch.cuda.device_count() + 7
    h = ctypes.c_void_p()
    assert lib.cola_create(ctypes.byref(h), ctypes.byref(p)) == b.COLA_ECUDA and not h.value
    assert b"cudaSetDevice" in lib.cola_last_error(None)
    torch.cuda.set_device(0)


@pytest.mark.faultinject
def test_a_faulting_kernel_surfaces_as_COLA_ECUDA(cola_mod):
    """COLA_ECUDA from a kernel fault, in a child process because the fault poisons its CUDA context: a workspace that is
    freed behind the library's back -- the kernels fault, the next synchronising call reports COLA_ECUDA with the CUDA
    message, and nothing hangs.  It raises an MMU fault on the GPU, so it is not part of the routine `-m gpu` run on a
    shared pool: select it with `-m faultinject`."""
    import subprocess
    import sys

    b = cola_mod
    child = r"""
import ctypes, sys, torch
sys.path.insert(0, %r)
from paper_2302_00850_b200 import binding as b, inputs
dims = (8, 8, 8, 16)
c = b.Cola(dims, 0.1245, 1.0)
ws = torch.empty(c.workspace_bytes(), dtype=torch.uint8, device="cuda")
c.set_workspace(ws)
c.gauge_upload(inputs.links_smooth(dims, 0.3, 9))
src = inputs.source_gaussian(dims, 5).cuda()
x, info = c.cg_solve(src, mixed=1)
assert info["converged"]
c._ws = None
del ws
torch.cuda.empty_cache()          # cudaFree: the library still holds the pointer
try:
    c.cg_solve(src, mixed=1)
except b.ColaError as ex:
    print("STATUS", ex.status, str(ex)[:120])
    sys.exit(0 if ex.status == b.COLA_ECUDA else 3)
print("no error raised")
sys.exit(4)
""" % os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", child], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, (r.returncode, r.stdout[-500:], r.stderr[-500:])
    assert "STATUS 2" in r.stdout
