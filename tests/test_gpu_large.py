"""Full-size parity at BASELINE.json configs 2, 3, 4 (32^3x64, 48^3x96, 64^3x128), in the launch configuration
bench.py times.  The oracle cannot sweep these lattices in seconds, so:
  * operators are compared on sampled output sites the oracle evaluates one by one (>= 4096 seeded random sites
    per parity, all 16 lattice corners, a strip of the boundary time-slices that exercises wrap and BC);
  * the 32^3x64 solve is compared with the stored oracle solve (tests/golden/solver_golden.json: iterations,
    sampled solution values, norm);
  * larger solves are checked through the residual b - M x evaluated by the ORACLE at sampled sites and through
    the global residual norm the library reports.
Links are generated on the GPU with the seeded generator (same integer hash as on the CPU, floating point equal
to rounding) and copied to the host for the oracle.
"""
import json
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = [pytest.mark.gpu, pytest.mark.large]
GOLD = os.path.join(os.path.dirname(__file__), "golden", "solver_golden.json")
TOL = {torch.float64: 1e-12, torch.float32: 2e-6}
EPS = {torch.float64: 2.0 ** -52, torch.float32: 2.0 ** -23}


def check_op(got, want, dtype):
    """relative L2 error at north_star's tolerance AND every real component within 64 eps of the largest one: on 10^4
    sampled sites a single component wrong by a per cent would move the norm by less than the fp32 tolerance."""
    assert rel(got, want) < TOL[dtype]
    assert np.abs(got - want).max() <= 64 * EPS[dtype] * np.abs(want).max()


def sample_sites(dims, n_random, seed):
    lx, ly, lz, lt = dims
    V = lx * ly * lz * lt
    rng = np.random.default_rng(seed)
    sites = set(int(s) for s in rng.integers(0, V, size=2 * n_random + 64))
    for cx in (0, lx - 1):
        for cy in (0, ly - 1):
            for cz in (0, lz - 1):
                for ct in (0, lt - 1):
                    sites.add(cx + lx * (cy + ly * (cz + lz * ct)))
    # a strip of both boundary time-slices (first x-y plane at z = 0 and z = Lz-1)
    for ct in (0, lt - 1):
        for cz in (0, lz - 1):
            base = lx * ly * (cz + lz * ct)
            sites.update(range(base, base + lx * ly))
    return np.array(sorted(sites), dtype=np.int64)


def parity_of(dims, sites):
    lx, ly, lz, lt = dims
    x = sites % lx
    y = (sites // lx) % ly
    z = (sites // (lx * ly)) % lz
    t = sites // (lx * ly * lz)
    return (x + y + z + t) & 1


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


class Big:
    def __init__(self, k):
        from paper_2302_00850_b200 import binding

        self.k = k
        self.cfg = inputs.CONFIGS[k]
        self.dims = self.cfg["dims"]
        U = inputs.make_links(k, device="cuda")
        # 64^3x128: carve what these tests use (no 8-real links, no 72-real fp32 A): 120 GB instead of 134 GB of workspace
        feats = (binding.COLA_FEAT_FULL_M | binding.COLA_FEAT_H16) if k == 4 else None
        self.ctx = binding.Cola(self.dims, self.cfg["kappa"], self.cfg["csw"], bc=inputs.BC, compress12=True, features=feats)
        self.ctx.gauge_upload(U)
        self.Un = U.cpu().numpy()
        del U
        torch.cuda.empty_cache()
        self.sites = sample_sites(self.dims, 4096, 7000 + k)
        self.par = parity_of(self.dims, self.sites)

    def close(self):
        self.ctx.close()
        torch.cuda.empty_cache()


@pytest.fixture(scope="module", params=[2, 3, 4])
def big(request):
    b = Big(request.param)
    yield b
    b.close()


def at_sites(canon, sites):
    return canon.reshape(-1, 4, 3)[torch.from_numpy(sites).to(canon.device)].cpu().numpy()


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_operators_on_sampled_sites(big, dtype):
    c, dims, cfg = big.ctx, big.dims, big.cfg
    assert len(big.sites) >= 8192 and (big.par == 0).sum() >= 4096 and (big.par == 1).sum() >= 4096
    psi = inputs.source_gaussian(dims, 4242 + big.k, device="cuda")
    psin = psi.cpu().numpy()
    ct = torch.complex128 if dtype == torch.float64 else torch.complex64
    internal = c.spinor_pack(psi.to(ct))
    args = (dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"])
    # full hopping term = the two parity dslashes
    out = torch.empty_like(internal)
    c.dslash_apply(0, internal[1], out=out[0])
    c.dslash_apply(1, internal[0], out=out[1])
    got = at_sites(c.spinor_unpack(out), big.sites)
    check_op(got, oracle.apply_sites(*args, "D", psin, big.sites), dtype)
    for which, dagger in (("M", False), ("Mdag", True)):
        got = at_sites(c.spinor_unpack(c.fermion_matrix_apply(internal, dagger=dagger)), big.sites)
        check_op(got, oracle.apply_sites(*args, which, psin, big.sites), dtype)
    even = big.sites[big.par == 0]
    for which, dagger in (("S", False), ("Sdag", True)):
        out.zero_()
        c.schur_apply(internal[0], dagger=dagger, out=out[0])
        got = at_sites(c.spinor_unpack(out), even)
        check_op(got, oracle.apply_sites(*args, which, psin, even), dtype)


def test_r8_operators_on_sampled_sites(big):
    """COLA_F32_R8 (8-real links + 48-real A) at full size, fp32 tolerance, and its solver mode."""
    c, dims, cfg = big.ctx, big.dims, big.cfg
    if big.k == 4:
        pytest.skip("64^3x128 context is carved without COLA_FEAT_R8 (workspace)")
    psi = inputs.source_gaussian(dims, 4343 + big.k, device="cuda")
    psin = psi.cpu().numpy()
    internal = c.spinor_pack(psi.to(torch.complex64))
    if c.gauge_info_r8() < 0.1:      # a link in the tail of the ensemble with |U00| < 0.1: the format is refused, not wrong
        from paper_2302_00850_b200 import binding
        with pytest.raises(binding.ColaError):
            c.fermion_matrix_apply(internal, fmt="r8")
        return
    args = (dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"])
    got = at_sites(c.spinor_unpack(c.fermion_matrix_apply(internal, fmt="r8")), big.sites)
    check_op(got, oracle.apply_sites(*args, "M", psin, big.sites), torch.float32)
    even = big.sites[big.par == 0]
    out = torch.zeros_like(internal)
    c.schur_apply(internal[0], dagger=True, out=out[0], fmt="r8")
    check_op(at_sites(c.spinor_unpack(out), even), oracle.apply_sites(*args, "Sdag", psin, even), torch.float32)
    if big.k == 2:
        b = inputs.source_gaussian(dims, inputs.config_seed_source(big.k), device="cuda")
        x, info = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=3)
        x1, info1 = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=1)
        assert info["converged"] and info["true_residual"] <= 1.05e-10
        assert abs(info["iters"] - info1["iters"]) <= 1 and info["reliable_updates"] == info1["reliable_updates"]


def test_mixed_precision_solve(big):
    c, dims, cfg, k = big.ctx, big.dims, big.cfg, big.k
    if cfg["source"] == "point":
        b = inputs.source_point(dims, 1, 2, device="cuda")        # one of BJ:c3's 12 spin-colour sources
    else:
        b = inputs.source_gaussian(dims, inputs.config_seed_source(k), device="cuda")
    x, info = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=True)
    assert info["converged"] and info["true_residual"] <= 1.05e-10 and info["reliable_updates"] >= 2
    # residual evaluated by the ORACLE at the sampled sites vs the library's own residual field there
    xn, bn = x.cpu().numpy(), b.cpu().numpy()
    Mx = oracle.apply_sites(dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"], "M", xn, big.sites)
    r_or = bn.reshape(-1, 4, 3)[big.sites] - Mx
    Mx_gpu = c.spinor_unpack(c.fermion_matrix_apply(c.spinor_pack(x)))
    r_gpu = at_sites(b - Mx_gpu, big.sites)
    bnorm = float(torch.linalg.vector_norm(b).item())
    # per-site residuals agree to fp64 rounding of the operator (|M x| ~ |b| locally)
    assert np.abs(r_or - r_gpu).max() <= 1e-12 * max(1.0, np.abs(Mx).max())
    # the sampled sites carry their share of a 1e-10 residual: rms over the sample extrapolated to the volume
    V = inputs.volume(dims)
    est = math.sqrt(float((np.abs(r_or) ** 2).sum()) * V / len(big.sites)) / bnorm
    if cfg["source"] != "point":
        assert est <= 3e-10
    glob = float(torch.linalg.vector_norm(b - Mx_gpu).item()) / bnorm
    assert abs(glob - info["true_residual"]) <= 1e-3 * glob + 1e-14
    if k == 2:
        g = json.load(open(GOLD))["2"]["eo"]
        assert abs(info["iters"] - g["iters"]) <= max(1, math.ceil(0.02 * g["iters"]))
        # SURVEY O8's schedule at full size: the passes after which the reliable updates fire follow from the stored
        # fp64 residual history of the ORACLE's solve (tests/schedule.py, pinned on the CPU against oracle.cgnr_mixed)
        from schedule import reliable_update_schedule

        want_upd, margin = reliable_update_schedule(g["history"], g["rmax0"], 0.1, 1e-10)
        xh, ih = c.cg_solve_history(b, tol=1e-10, even_odd=True, mixed=True)
        assert ih["reliable_updates"] == info["reliable_updates"] and torch.equal(xh, x)
        h = np.asarray(ih["history"])
        n = min(len(h), len(g["history"]))
        assert np.max(np.abs(h[:n] - np.asarray(g["history"])[:n]) / np.asarray(g["history"])[:n]) < 1e-4
        if margin > 1e-3:
            assert ih["update_iters"] == want_upd, (ih["update_iters"], want_upd)
        xs = xn.reshape(-1, 12)[np.array(g["sites"])]
        want = np.array(g["x_re"]) + 1j * np.array(g["x_im"])
        assert np.linalg.norm(xs - want) / np.linalg.norm(want) < 5e-8
        assert abs(np.linalg.norm(xn.ravel()) - g["x_norm"]) / g["x_norm"] < 1e-8
        # pure fp64 solve: same count
        x64, info64 = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=False)
        assert info64["converged"] and abs(info64["iters"] - g["iters"]) <= max(1, math.ceil(0.02 * g["iters"]))
        assert rel(x64.cpu().numpy(), xn) < 5e-9


def test_16bit_operator_and_solver_at_full_size(big):
    """COLA_F32_H16 in bench.py's launch configuration: sampled-site operator parity within the
    storage-error tolerance of tests/test_gpu_h16.py, and the mixed = 2 solve to the same bar as mixed = 1."""
    c, dims, cfg, k = big.ctx, big.dims, big.cfg, big.k
    psi = inputs.source_gaussian(dims, 4342 + k, device="cuda")
    psin = psi.cpu().numpy()
    internal = c.spinor_pack(psi.to(torch.complex64))
    args = (dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"])
    got = at_sites(c.spinor_unpack(c.fermion_matrix_apply(internal, h16=True)), big.sites)
    e = rel(got, oracle.apply_sites(*args, "M", psin, big.sites))
    assert 1e-6 < e < 5e-4, e
    even = big.sites[big.par == 0]
    out = torch.zeros_like(internal)
    c.schur_apply(internal[0], dagger=True, out=out[0], h16=True)
    assert rel(at_sites(c.spinor_unpack(out), even), oracle.apply_sites(*args, "Sdag", psin, even)) < 5e-4
    if k == 4:
        return      # the 64^3x128 solve is covered by test_mixed_precision_solve; keep this test short
    b = inputs.source_point(dims, 1, 2, device="cuda") if cfg["source"] == "point" else inputs.source_gaussian(dims, inputs.config_seed_source(k), device="cuda")
    x, info = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=2)
    assert info["converged"] and info["true_residual"] <= 1.05e-10
    x1, info1 = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=1)
    assert abs(info["iters"] - info1["iters"]) <= max(1, math.ceil(0.02 * info1["iters"])), (info["iters"], info1["iters"])
    assert rel(x.cpu().numpy(), x1.cpu().numpy()) < 5e-9
    if k == 2:
        g = json.load(open(GOLD))["2"]["eo"]
        assert abs(info["iters"] - g["iters"]) <= max(1, math.ceil(0.02 * g["iters"]))
        xs = x.cpu().numpy().reshape(-1, 12)[np.array(g["sites"])]
        want = np.array(g["x_re"]) + 1j * np.array(g["x_im"])
        assert np.linalg.norm(xs - want) / np.linalg.norm(want) < 5e-8


def test_multi_rhs_operators_at_full_size(big):
    """Multi-rhs launches at full size: 3 vectors (a ragged last rhs group; 2 at 64^3x128),
    sampled-site parity against the oracle for one of them and bit-identity with the single-rhs kernels for all."""
    c, dims, cfg, k = big.ctx, big.dims, big.cfg, big.k
    nv = 2 if k == 4 else 3                          # 64^3x128: two vectors keep the test inside 180 GB beside the 123 GB workspace
    c.set_mrhs_workspace(nv, for_solver=False)      # operators only: 1.5 fp64 half vectors per right-hand side
    full = []
    for n in range(nv):
        p = inputs.source_gaussian(dims, 4442 + k + n, device="cuda")
        full.append(c.spinor_pack(p.to(torch.complex64)))
        if n == nv - 1:
            last = p.cpu().numpy()
        del p
    full = torch.stack(full)
    torch.cuda.empty_cache()
    out = c.fermion_matrix_apply_mrhs(full)
    args = (dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"])
    got = at_sites(c.spinor_unpack(out[nv - 1].contiguous()), big.sites)
    check_op(got, oracle.apply_sites(*args, "M", last, big.sites), torch.float32)
    del got
    outs = c.schur_apply_mrhs(full[:, 0].contiguous(), dagger=True)
    for n in range(nv):
        assert torch.equal(out[n], c.fermion_matrix_apply(full[n].contiguous()))
        assert torch.equal(outs[n], c.schur_apply(full[n, 0].contiguous(), dagger=True))
    c.release_mrhs_workspace()
    torch.cuda.empty_cache()


def oracle_checked_residual(big, b, x, info, note):
    """b - M x evaluated by the ORACLE at the sampled sites against the library's residual field there, and the
    library's reported true residual against the norm of that field (as test_mixed_precision_solve)."""
    c, dims, cfg = big.ctx, big.dims, big.cfg
    assert info["converged"] and info["true_residual"] <= 1.05e-10, (note, info)
    # the oracle reads x only at the sampled sites and their neighbours: hand it the full array (host copy)
    xn = x.cpu().numpy()
    Mx = oracle.apply_sites(dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"], "M", xn, big.sites)
    del xn
    Mx_gpu = c.spinor_unpack(c.fermion_matrix_apply(c.spinor_pack(x)))
    r_gpu_field = b - Mx_gpu
    r_or = at_sites(b, big.sites) - Mx
    r_gpu = at_sites(r_gpu_field, big.sites)
    assert np.abs(r_or - r_gpu).max() <= 1e-12 * max(1.0, np.abs(Mx).max()), note
    bnorm = float(torch.linalg.vector_norm(b).item())
    glob = float(torch.linalg.vector_norm(r_gpu_field).item()) / bnorm
    assert glob <= 1.05e-10 and abs(glob - info["true_residual"]) <= 1e-3 * glob + 1e-14, (note, glob, info["true_residual"])
    del Mx_gpu, r_gpu_field
    torch.cuda.empty_cache()


def config_source(big, n=None):
    dims, cfg, k = big.dims, big.cfg, big.k
    if n is not None:
        return inputs.source_point(dims, n % 4, n % 3, device="cuda")
    if cfg["source"] == "point":
        return inputs.source_point(dims, 1, 2, device="cuda")
    return inputs.source_gaussian(dims, inputs.config_seed_source(k), device="cuda")


@pytest.mark.parametrize("mixed", [1, 2])
def test_bicgstab_at_full_size(big, mixed):
    """BiCGStab on the Schur system in bench.py's launch configuration.  At these sizes the
    reductions of its BLAS-1 kernels and of the <t, s> fused into the operator kernel (grid_sum_last_n) span many groups
    of 256 blocks, a path the small lattices of test_gpu_bicgstab.py never take.  The solution is held to the oracle
    through b - M x at the sampled sites; at 32^3x64 also to the stored solution of the ORACLE's CGNR solve."""
    c, dims, k = big.ctx, big.dims, big.k
    b = config_source(big)
    x, info = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=mixed, method="bicgstab")
    assert info["reliable_updates"] >= 1
    oracle_checked_residual(big, b, x, info, ("bicgstab", k, mixed))
    xc, infoc = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=mixed)
    assert info["iters"] < infoc["iters"]                     # two S per pass against S and S^+, and fewer passes
    assert rel(x.cpu().numpy(), xc.cpu().numpy()) < 5e-9
    if k == 2:
        g = json.load(open(GOLD))["2"]["eo"]
        xs = x.cpu().numpy().reshape(-1, 12)[np.array(g["sites"])]
        want = np.array(g["x_re"]) + 1j * np.array(g["x_im"])
        assert np.linalg.norm(xs - want) / np.linalg.norm(want) < 5e-8


@pytest.mark.parametrize("method", ["cgnr", "bicgstab"])
def test_batched_solvers_at_full_size(big, method):
    """cola_cg_solve_mrhs with 4 point sources at 32^3x64 and 48^3x96: the multi-rhs launches inside
    a solve (z-banded sweep, per-system reductions over many block groups).  Each system: oracle-sampled residual, pass
    count and solution against the sequential solver of the same system."""
    c, dims, k = big.ctx, big.dims, big.k
    if k == 4:
        pytest.skip("64^3x128: the batched solver's workspace does not fit beside the 120 GB context")
    nrhs = 4
    c.set_mrhs_workspace(nrhs, for_solver=True)
    srcs = [config_source(big, n) for n in range(nrhs)]
    x, infos = c.cg_solve_mrhs(torch.stack(srcs), tol=1e-10, mixed=1, method=method)
    for n in range(nrhs):
        xs, info = c.cg_solve(srcs[n], tol=1e-10, even_odd=True, mixed=1, method=method)
        if method == "cgnr":
            assert abs(info["iters"] - infos[n]["iters"]) <= 1 and info["reliable_updates"] == infos[n]["reliable_updates"], (n, info, infos[n])
        else:
            assert abs(info["iters"] - infos[n]["iters"]) <= max(2, math.ceil(0.1 * info["iters"])), (n, info, infos[n])
        assert rel(x[n].cpu().numpy(), xs.cpu().numpy()) < 5e-9
        if n in (0, nrhs - 1):
            oracle_checked_residual(big, srcs[n], x[n].contiguous(), infos[n], (method, k, n))
        else:
            assert infos[n]["converged"] and infos[n]["true_residual"] <= 1.05e-10
    c.release_mrhs_workspace()
    torch.cuda.empty_cache()


def test_low_modes_and_deflated_start_at_full_size(big):
    """cola_eig_lowest + cola_cg_solve_deflated at 32^3x64: the returned pairs satisfy H u = lambda u with H = S^+S applied
    by the ORACLE at sampled even sites, and the deflated solve reaches the stored oracle solution."""
    c, dims, cfg, k = big.ctx, big.dims, big.cfg, big.k
    if k != 2:
        pytest.skip("low modes: 32^3x64 only (DESIGN.md section 7)")
    n_ev = 8                                                 # bench.py's low_modes configuration
    ev, evecs, info = c.eig_lowest(n_ev, tol=1e-9)
    assert info["converged"], info
    ev = np.asarray(ev)
    assert np.all(ev > 0) and np.all(np.diff(ev) >= 0) and max(info["residuals"]) < 1e-6 * info["cheb_hi"]
    even = big.sites[big.par == 0]
    args = (dims, inputs.BC, big.Un, cfg["kappa"], cfg["csw"])
    full = torch.zeros((2, 12, c.Vh, 2), dtype=torch.float64, device="cuda")
    for i in (0, n_ev - 1):
        full[0] = evecs[i]
        u = c.spinor_unpack(full)
        Su = torch.zeros_like(full)
        c.schur_apply(full[0], out=Su[0])                                    # S u on the GPU (fp64, oracle-verified above) ...
        Su_c = c.spinor_unpack(Su)
        Hu = oracle.apply_sites(*args, "Sdag", Su_c.cpu().numpy(), even)     # ... S^+ (S u) by the oracle at the sampled sites
        Su_or = oracle.apply_sites(*args, "S", u.cpu().numpy(), even)
        assert rel(at_sites(Su_c, even), Su_or) < 1e-12
        lhs = Hu - ev[i] * at_sites(u, even)
        # the sample's share of the residual cannot exceed the whole (|H u - lambda u| over all even sites, |u| = 1)
        assert np.linalg.norm(lhs) <= info["residuals"][i] * (1 + 1e-6) + 1e-11, (i, np.linalg.norm(lhs), info["residuals"][i])
        assert np.linalg.norm(at_sites(u, even)) > 0
    b = config_source(big)
    x0, i0 = c.cg_solve(b, tol=1e-10, even_odd=True, mixed=1)
    x1, i1 = c.cg_solve_deflated(b, ev, evecs, tol=1e-10, mixed=1)
    assert i1["converged"] and i1["true_residual"] <= 1.05e-10 and i1["iters"] <= i0["iters"]
    g = json.load(open(GOLD))["2"]["eo"]
    xs = x1.cpu().numpy().reshape(-1, 12)[np.array(g["sites"])]
    want = np.array(g["x_re"]) + 1j * np.array(g["x_im"])
    assert np.linalg.norm(xs - want) / np.linalg.norm(want) < 5e-8
