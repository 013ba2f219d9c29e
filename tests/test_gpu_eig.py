"""Low modes of S^+ S (cola_eig_lowest) against the oracle's definition (oracle.lowest_modes:
dense Hermitian eigen-solve on small lattices, ARPACK on the oracle's operator above; pinned on the CPU against the
brute-force dense Schur complement), and the deflated start of the CGNR solver."""
import numpy as np
import pytest
import torch

import oracle
from paper_2302_00850_b200 import inputs

pytestmark = pytest.mark.gpu
BC = (1, 1, 1, -1)


def setup(dims, kappa=0.1245, csw=1.0, seed=7):
    from paper_2302_00850_b200 import binding

    U = inputs.links_smooth(dims, 0.3, seed)
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    c = binding.Cola(dims, kappa, csw, bc=BC)
    c.gauge_upload(U)
    return c, Un, A, Ainv, kappa


@pytest.mark.parametrize("dims,n_ev", [((4, 2, 2, 4), 6), ((4, 4, 4, 4), 8), ((8, 8, 8, 16), 8)])
def test_lowest_modes_match_the_oracle(dims, n_ev):
    c, Un, A, Ainv, kappa = setup(dims)
    want, want_vecs = oracle.lowest_modes(dims, BC, Un, A, Ainv, kappa, n_ev + 2)
    ev, evecs, info = c.eig_lowest(n_ev, tol=1e-11)
    assert info["converged"], info
    ev = np.asarray(ev)
    assert np.all(np.diff(ev) >= 0)
    assert np.max(np.abs(ev - want[:n_ev]) / want[:n_ev]) < 1e-8, (ev, want[:n_ev])
    assert max(info["residuals"]) < 1e-7 * info["cheb_hi"]
    # eigenvectors: unpack to canonical arrays, check H v = lambda v with the ORACLE's operator, orthonormality, and the
    # overlap with the oracle's eigenspace (eigenvalues closer than 1e-6 relative are treated as one space)
    full = torch.zeros((2, 12, c.Vh, 2), dtype=torch.float64, device="cuda")
    vs = []
    for i in range(n_ev):
        full[0] = evecs[i]
        vs.append(c.spinor_unpack(full).cpu().numpy())
    G = np.array([[np.vdot(a.ravel(), b.ravel()) for b in vs] for a in vs])
    assert np.abs(G - np.eye(n_ev)).max() < 1e-9
    for i in (0, n_ev - 1):
        Hv = oracle.schur(dims, BC, Un, A, Ainv, kappa, oracle.schur(dims, BC, Un, A, Ainv, kappa, vs[i]), dagger=True)
        assert np.linalg.norm((Hv - ev[i] * vs[i]).ravel()) < 1e-7 * info["cheb_hi"]
    W = want_vecs.reshape(n_ev + 2, -1)
    for i in range(n_ev):
        near = np.abs(want - ev[i]) < 1e-6 * ev[i] + 0.5 * min(np.diff(want).min(), 1e9) * 0  # same eigenvalue
        near |= np.abs(want - ev[i]) / ev[i] < 1e-6
        proj = sum(abs(np.vdot(W[j], vs[i].ravel())) ** 2 for j in np.flatnonzero(near))
        assert abs(proj - 1) < 1e-6, (i, proj)
    c.close()


def test_a_wrong_filter_window_is_detected_and_corrected():
    """The filter amplifies what lies below cheb_lo; the n_ev largest Ritz pairs of the filtered operator are the n_ev lowest
    modes of H only if at least n_ev eigenvalues lie below cheb_lo and none above cheb_hi (an even-order Chebyshev
    polynomial amplifies those as well).  Converged pairs from a wrong window have small residuals, so only the check of
    the returned eigenvalues against the window tells; the library then corrects the window and repeats."""
    dims, n_ev = (4, 4, 4, 4), 8
    c, Un, A, Ainv, kappa = setup(dims)
    want, _ = oracle.lowest_modes(dims, BC, Un, A, Ainv, kappa, n_ev + 2)
    # (a) only two eigenvalues below cheb_lo, eight wanted
    lo_req = 0.5 * (want[1] + want[2])
    ev, _, info = c.eig_lowest(n_ev, tol=1e-11, cheb_lo=lo_req)
    assert info["converged"] and info["cheb_lo"] > want[n_ev - 1] > lo_req, info
    assert np.max(np.abs(np.asarray(ev) - want[:n_ev]) / want[:n_ev]) < 1e-8, (ev, want[:n_ev])
    # (b) the upper edge below the top of the spectrum: the top modes come out first, are recognised, the edge is moved
    ev0, _, info0 = c.eig_lowest(n_ev, tol=1e-11)
    hi_req = 0.5 * info0["cheb_hi"] / 1.15
    ev, _, info = c.eig_lowest(n_ev, tol=1e-11, cheb_hi=hi_req, cheb_lo=min(2.0 * want[n_ev], 0.5 * hi_req))
    assert info["converged"] and info["cheb_hi"] > hi_req, info
    assert np.max(np.abs(np.asarray(ev) - want[:n_ev]) / want[:n_ev]) < 1e-8, (ev, want[:n_ev])
    assert info["op_applications"] > info0["op_applications"]          # the discarded run is accounted for
    c.close()


def test_plain_lanczos_and_parameter_checks():
    dims = (4, 4, 4, 4)
    c, Un, A, Ainv, kappa = setup(dims)
    want, _ = oracle.lowest_modes(dims, BC, Un, A, Ainv, kappa, 4)
    # order 1 = plain Lanczos on -H: slower, same answer
    ev, evecs, info = c.eig_lowest(4, n_kr=40, cheb_order=1, tol=1e-9, max_restarts=400)
    assert info["converged"] and np.max(np.abs(np.asarray(ev) - want) / want) < 1e-7
    ev2, _, info2 = c.eig_lowest(4, tol=1e-11)
    assert info2["op_applications"] > 0 and np.max(np.abs(np.asarray(ev2) - want) / want) < 1e-8
    from paper_2302_00850_b200 import binding as b
    for kw in (dict(n_ev=0), dict(n_ev=33), dict(n_ev=8, n_kr=9)):
        with pytest.raises((b.ColaError, ValueError)):
            c.eig_lowest(**kw)
    # max_restarts reached: COLA_ENOCONV, results of the last restart returned
    ev3, _, info3 = c.eig_lowest(4, n_kr=8, cheb_order=1, max_restarts=1, tol=1e-14)
    assert not info3["converged"] and info3["restarts"] == 1 and all(np.isfinite(ev3))
    c.close()


def test_deflated_start_saves_iterations_and_gives_the_same_solution():
    dims = (8, 8, 8, 16)
    c, Un, A, Ainv, kappa = setup(dims, kappa=0.1265)      # lighter quark: the low modes matter
    b = inputs.source_gaussian(dims, 41)
    ev, evecs, info = c.eig_lowest(16, tol=1e-9)
    assert info["converged"]
    ref = oracle.cgnr(dims, BC, Un, A, Ainv, kappa, b.numpy(), even_odd=True, tol=1e-10)
    for mixed in (0, 1):
        x0, i0 = c.cg_solve(b.cuda(), mixed=mixed)
        x1, i1 = c.cg_solve_deflated(b.cuda(), ev, evecs, mixed=mixed)
        assert i0["converged"] and i1["converged"] and i1["true_residual"] <= 1.05e-10
        assert i1["iters"] < i0["iters"], (i1["iters"], i0["iters"])
        for x in (x0, x1):
            xn = x.cpu().numpy()
            assert np.linalg.norm((xn - ref["x"]).ravel()) / np.linalg.norm(ref["x"].ravel()) < 5e-9
            res = np.linalg.norm((b.numpy() - oracle.M(dims, BC, Un, A, kappa, xn)).ravel()) / np.linalg.norm(b.numpy().ravel())
            assert res <= 1.05e-10
    c.close()
