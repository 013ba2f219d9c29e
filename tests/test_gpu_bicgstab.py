"""BiCGStab on the Schur complement (cola_solve_params.method = COLA_BICGSTAB) against the
oracle's BiCGStab (oracle/cola_oracle.c, pinned on the CPU against the dense inverse, CGNR's solution and scipy's
implementation): solution, fp64 true residual recomputed with the ORACLE's M, pass counts, and the residual history
pass by pass in fp64 mode."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu
BC = (1, 1, 1, -1)


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.mark.parametrize("dims,kind", [((2, 2, 2, 2), "haar"), ((4, 4, 4, 4), "haar"), ((12, 10, 6, 4), "smooth"), ((8, 8, 8, 16), "smooth"),
                                       ((16, 16, 16, 32), "smooth")])   # 65 536 even sites: every reduction spans 4 groups of 256 blocks
def test_bicgstab_matches_the_oracle(dims, kind):
    from paper_2302_00850_b200 import binding

    kappa, csw = (0.12, 1.0) if kind == "haar" else (0.1245, 1.0)
    U = inputs.links_haar(dims, 5) if kind == "haar" else inputs.links_smooth(dims, 0.3, 5)
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = inputs.source_gaussian(dims, 21)
    bn = b.numpy()
    ref = oracle.bicgstab(dims, BC, Un, A, Ainv, kappa, bn, even_odd=True, tol=1e-10)
    assert ref["converged"]
    cg = oracle.cgnr(dims, BC, Un, A, Ainv, kappa, bn, even_odd=True, tol=1e-10)
    c = binding.Cola(dims, kappa, csw, bc=BC)
    c.gauge_upload(U)
    # mixed = 3 (8-real links) is offered for the smooth ensembles only: Haar links have |U00| < 0.1 somewhere
    for mixed in (0, 1, 2) + ((3,) if kind == "smooth" else ()):
        x, info = c.cg_solve_history(b.cuda(), tol=1e-10, even_odd=True, mixed=mixed, method="bicgstab")
        assert info["converged"] and info["true_residual"] <= 1.05e-10, (mixed, info)
        xn = x.cpu().numpy()
        res = np.linalg.norm((bn - oracle.M(dims, BC, Un, A, kappa, xn)).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10 and abs(res - info["true_residual"]) <= 1e-3 * res + 1e-14
        assert rel(xn, ref["x"]) < 5e-9 and rel(xn, cg["x"]) < 5e-9
        h, h_ref = np.asarray(info["history"]), np.asarray(ref["history"])
        if mixed == 0:
            # fp64: the same recurrence; rounding differences are amplified along the non-monotone BiCGStab history, so
            # the first passes agree to rounding, and the count within max(1, 2 %)
            assert abs(info["iters"] - ref["iters"]) <= max(1, math.ceil(0.02 * ref["iters"])), (info["iters"], ref["iters"])
            n = min(6, len(h), len(h_ref))
            assert np.max(np.abs(h[:n] - h_ref[:n]) / h_ref[:n]) < 1e-9
        else:
            # fp32 / 16-bit inner passes: BiCGStab's count is sensitive to rounding; hold it to the oracle's within 15 %
            # (+2), and well below CGNR's
            assert abs(info["iters"] - ref["iters"]) <= max(2, math.ceil(0.15 * ref["iters"])), (mixed, info["iters"], ref["iters"])
            assert info["reliable_updates"] >= 1
        if min(dims) > 2:
            assert info["iters"] < cg["iters"]
    # host buffers, and the same answer
    xh, ih = c.cg_solve(b.pin_memory(), tol=1e-10, even_odd=True, mixed=1, method="bicgstab")
    x1, i1 = c.cg_solve(b.cuda(), tol=1e-10, even_odd=True, mixed=1, method="bicgstab")
    assert ih["iters"] == i1["iters"] and rel(xh.numpy(), x1.cpu().numpy()) < 1e-12
    # not offered on the unpreconditioned system, nor batched
    with pytest.raises(binding.ColaError) as e:
        c.cg_solve(b.cuda(), even_odd=False, method="bicgstab")
    assert e.value.status == binding.COLA_EINVAL
    xx, info = c.cg_solve(b.cuda(), max_iter=2, method="bicgstab", mixed=1)
    assert not info["converged"] and info["iters"] == 2 and 0 < info["true_residual"] < 1
    c.close()


@pytest.mark.parametrize("mixed", [1, 2, 3])
def test_batched_bicgstab_matches_the_oracle_and_the_sequential_solver(mixed):
    """cola_cg_solve_mrhs with method = COLA_BICGSTAB: every system's solution against the oracle (true residual with the
    ORACLE's M, solution against oracle.cgnr's), pass counts against the sequential CUDA BiCGStab of the same system
    (the recurrences differ only in the summation order of the fused |t|^2) and against the oracle's BiCGStab."""
    from paper_2302_00850_b200 import binding

    dims, kappa, csw = (8, 8, 8, 16), 0.1245, 1.0
    U = inputs.links_smooth(dims, 0.3, 33)
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    c = binding.Cola(dims, kappa, csw, bc=BC)
    c.gauge_upload(U)
    srcs = [inputs.source_point(dims, s, s % 3) for s in range(4)] + [inputs.source_gaussian(dims, 66), torch.zeros_like(inputs.source_gaussian(dims, 1))]
    x, infos = c.cg_solve_mrhs(torch.stack(srcs).cuda(), tol=1e-10, mixed=mixed, method="bicgstab")
    for n, s in enumerate(srcs[:-1]):
        bn = s.numpy()
        xn = x[n].cpu().numpy()
        res = np.linalg.norm((bn - oracle.M(dims, BC, Un, A, kappa, xn)).ravel()) / np.linalg.norm(bn.ravel())
        assert res <= 1.05e-10 and infos[n]["true_residual"] <= 1.05e-10, (n, res, infos[n])
        assert infos[n]["reliable_updates"] >= 1
        x1, i1 = c.cg_solve(s.cuda(), tol=1e-10, even_odd=True, mixed=mixed, method="bicgstab")
        assert abs(infos[n]["iters"] - i1["iters"]) <= max(2, math.ceil(0.1 * i1["iters"])), (n, infos[n]["iters"], i1["iters"])
        assert rel(xn, x1.cpu().numpy()) < 5e-9
        if n in (0, 4):
            ref = oracle.bicgstab(dims, BC, Un, A, Ainv, kappa, bn, even_odd=True, tol=1e-10)
            cg = oracle.cgnr(dims, BC, Un, A, Ainv, kappa, bn, even_odd=True, tol=1e-10)
            assert rel(xn, ref["x"]) < 5e-9 and rel(xn, cg["x"]) < 5e-9
            assert abs(infos[n]["iters"] - ref["iters"]) <= max(2, math.ceil(0.15 * ref["iters"])), (infos[n]["iters"], ref["iters"])
            assert infos[n]["iters"] < cg["iters"]
    # the zero source: solution zero, no passes
    assert infos[-1]["iters"] == 0 and float(x[-1].abs().max()) == 0.0
    # max_iter: COLA_ENOCONV, the last iterates returned with their true residuals
    xx, inf2 = c.cg_solve_mrhs(torch.stack(srcs[:3]).cuda(), tol=1e-10, mixed=mixed, method="bicgstab", max_iter=3)
    assert all(i["iters"] == 3 and not i["converged"] and 0 < i["true_residual"] < 1 for i in inf2)
    c.close()


@pytest.mark.parametrize("mixed", [0, 1])
def test_exact_convergence_at_the_half_step_is_not_a_breakdown(mixed):
    """Unit links (A = 1), periodic boundaries, source psi(x) = (-1)^(x+y) chi: the hops in x and y cancel those in z and t,
    D psi = 0 exactly in floating point, so S psi_e = psi_e, alpha = 1, s = r - alpha v = 0 and t = S s = 0 in the first pass.
    omega = <t, s> / <t, t> is 0/0 there; the solver must finish with x = x + alpha p (= b) instead of reporting NaN.  The
    same source in a batch must not disturb its neighbours."""
    from paper_2302_00850_b200 import binding

    dims, kappa, bc = (4, 4, 4, 8), 0.1, (1, 1, 1, 1)      # kappa below the free-field critical value 1/8: M is regular
    U = inputs.links_unit(dims)
    c = binding.Cola(dims, kappa, 1.0, bc=bc)
    c.gauge_upload(U)
    lx, ly, lz, lt = dims
    sign = (-1.0) ** (np.arange(lx)[None, None, None, :] + np.arange(ly)[None, None, :, None]) * np.ones((lt, lz, 1, 1))
    chi = (np.arange(12).reshape(4, 3) - 5.0) + 1j * (np.arange(12).reshape(4, 3) % 4)
    b = torch.from_numpy(sign[..., None, None] * chi).to(torch.complex128)
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, 1.0)
    assert np.abs(oracle.M(dims, bc, Un, A, kappa, b.numpy()) - b.numpy()).max() == 0.0     # M b = b: the solution is b
    x, info = c.cg_solve(b.cuda(), tol=1e-10, even_odd=True, mixed=mixed, method="bicgstab")
    assert info["converged"] and info["iters"] == 1 and info["true_residual"] == 0.0, info
    assert torch.equal(x.cpu(), b)
    if mixed:
        g = inputs.source_gaussian(dims, 9)
        xs, infos = c.cg_solve_mrhs(torch.stack([g, b, 2 * g]).cuda(), tol=1e-10, mixed=1, method="bicgstab")
        assert all(i["converged"] and i["true_residual"] <= 1.05e-10 for i in infos), infos
        assert torch.equal(xs[1].cpu(), b) and infos[1]["iters"] == 1
        assert rel(xs[2].cpu().numpy(), 2 * xs[0].cpu().numpy()) < 1e-9
    c.close()
