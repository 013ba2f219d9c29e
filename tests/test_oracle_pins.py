"""Pins of the CPU oracle against what the physics and the mathematics fix (SURVEY.md §8(c) "Pins").

The paper prints no worked example (PAPER.md has no equations or numbers), so every pin is a closed
form, an invariant or an independent brute force.  CPU only.
"""
import numpy as np
import pytest
import torch

import bruteforce as bf
import oracle
from paper_2302_00850_b200 import inputs

BC = (1, 1, 1, -1)


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def np_links(kind, dims, seed=7, eps=0.3):
    if kind == "haar":
        return inputs.links_haar(dims, seed).numpy()
    if kind == "smooth":
        return inputs.links_smooth(dims, eps, seed).numpy()
    return inputs.links_unit(dims).numpy()


def rand_spinor(dims, seed):
    return inputs.source_gaussian(dims, seed).numpy()


# ---------------------------------------------------------------------------------------------
# O2: gamma algebra
# ---------------------------------------------------------------------------------------------
def test_gamma_matrices_match_hand_typed_and_clifford():
    g = oracle.gamma()
    for mu in range(4):
        assert np.array_equal(g[mu], bf.GAMMA[mu])
        assert np.array_equal(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=0)
    assert np.array_equal(g[4], bf.GAMMA5)
    assert np.array_equal(g[4], g[0] @ g[1] @ g[2] @ g[3])


def test_sigma_matches_closed_form_blocks():
    s = oracle.sigma()
    for (mu, nu), ref in bf.SIGMA.items():
        assert np.allclose(s[mu, nu], ref, atol=1e-16)
        assert np.allclose(s[nu, mu], -ref, atol=1e-16)
    for mu in range(4):
        assert np.allclose(s[mu, mu], 0)


# ---------------------------------------------------------------------------------------------
# Pin 1: free field, closed form on every momentum (O1, O2, O3, BC, kappa normalisation)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,bc", [((4, 4, 4, 4), BC), ((4, 2, 6, 4), BC), ((4, 4, 2, 2), (1, -1, 1, 1))])
def test_free_field_plane_waves(dims, bc):
    kappa, csw = 0.12, 1.3   # csw arbitrary: F = 0 on unit links
    lx, ly, lz, lt = dims
    U = np_links("unit", dims)
    A = oracle.clover(dims, U, kappa, csw)
    assert np.allclose(A, np.eye(12), atol=1e-15)
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    coords = [x, y, z, t]
    rng = np.random.default_rng(1)
    worst = 0.0
    for n in np.ndindex(lx, ly, lz, lt):
        p = [(2 * np.pi * n[mu] / dims[mu]) if bc[mu] == 1 else ((2 * n[mu] + 1) * np.pi / dims[mu]) for mu in range(4)]
        chi = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        phase = np.exp(1j * sum(p[mu] * coords[mu] for mu in range(4)))
        psi = phase[..., None, None] * chi
        Mp = (1 - 2 * kappa * sum(np.cos(p))) * np.eye(4) + 2j * kappa * sum(np.sin(p[mu]) * bf.GAMMA[mu] for mu in range(4))
        expect = phase[..., None, None] * (Mp @ chi)
        got = oracle.M(dims, bc, U, A, kappa, psi)
        worst = max(worst, rel(got, expect))
        # eigenvalues of M(p): 1 - 2k sum cos +- 2ik sqrt(sum sin^2), each doubly degenerate in spin
        lam = np.linalg.eigvals(Mp)
        s = 2 * kappa * np.sqrt(sum(np.sin(p) ** 2))
        ref = 1 - 2 * kappa * sum(np.cos(p))
        assert np.allclose(np.sort(lam.imag), np.sort([-s, -s, s, s]), atol=1e-12)
        assert np.allclose(lam.real, ref, atol=1e-12)
    assert worst < 1e-13


# ---------------------------------------------------------------------------------------------
# Pin 2: gamma5-hermiticity (signs of forward/backward hops, U vs U^dagger, hermiticity of A)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_gamma5_hermiticity_M_and_schur(kind):
    dims, kappa, csw = (4, 4, 2, 6), 0.124, 1.1
    U = np_links(kind, dims)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    a, b = rand_spinor(dims, 11), rand_spinor(dims, 12)
    lhs = np.vdot(a, oracle.M(dims, BC, U, A, kappa, b))
    rhs = np.vdot(oracle.M(dims, BC, U, A, kappa, a, dagger=True), b)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    mask = (oracle.parity_mask(dims) == 0)[..., None, None]
    ae, be = a * mask, b * mask
    lhs = np.vdot(ae, oracle.schur(dims, BC, U, A, Ainv, kappa, be))
    rhs = np.vdot(oracle.schur(dims, BC, U, A, Ainv, kappa, ae, dagger=True), be)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


# ---------------------------------------------------------------------------------------------
# Pin 3: gauge covariance (link placement/orientation in O3 and every leaf of O4)
# ---------------------------------------------------------------------------------------------
def test_gauge_covariance():
    dims, kappa, csw = (4, 4, 4, 2), 0.12, 1.0
    U = inputs.links_haar(dims, 21)
    g = inputs.su3_site_field(dims, 22)
    psi = inputs.source_gaussian(dims, 23)
    Ug = inputs.gauge_transform_links(U, g).numpy()
    psig = inputs.gauge_transform_spinor(psi, g).numpy()
    A = oracle.clover(dims, U.numpy(), kappa, csw)
    Ag = oracle.clover(dims, Ug, kappa, csw)
    out = oracle.M(dims, BC, U.numpy(), A, kappa, psi.numpy())
    outg = oracle.M(dims, BC, Ug, Ag, kappa, psig)
    expect = inputs.gauge_transform_spinor(torch.from_numpy(out), g).numpy()
    assert rel(outg, expect) < 1e-13
    # the clover block itself transforms as (1 (x) g) A (1 (x) g^dagger)
    gn = g.numpy()
    G12 = np.einsum("st,...ab->...satb", np.eye(4), gn).reshape(gn.shape[:4] + (12, 12))
    assert rel(Ag, G12 @ A @ bf.dag(G12)) < 1e-13


# ---------------------------------------------------------------------------------------------
# Pin 4: pure gauge = transformed free field (closed form through non-trivial links and the BC)
# ---------------------------------------------------------------------------------------------
def test_pure_gauge_is_transformed_free_field():
    dims, kappa, csw = (4, 4, 2, 4), 0.118, 1.0
    g = inputs.su3_site_field(dims, 31)
    U = inputs.gauge_transform_links(inputs.links_unit(dims), g).numpy()
    A = oracle.clover(dims, U, kappa, csw)
    assert np.allclose(A, np.eye(12), atol=1e-14)
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    p = [2 * np.pi * 1 / lx, 2 * np.pi * 3 / ly, 0.0, 3 * np.pi / lt]
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    chi = np.arange(12).reshape(4, 3) * (0.3 - 0.1j) + 1.0
    Mp = (1 - 2 * kappa * sum(np.cos(p))) * np.eye(4) + 2j * kappa * sum(np.sin(p[mu]) * bf.GAMMA[mu] for mu in range(4))
    psi = torch.from_numpy(phase[..., None, None] * chi)
    expect = inputs.gauge_transform_spinor(torch.from_numpy(phase[..., None, None] * (Mp @ chi)), g).numpy()
    got = oracle.M(dims, BC, U, A, kappa, inputs.gauge_transform_spinor(psi, g).numpy())
    assert rel(got, expect) < 1e-13


# ---------------------------------------------------------------------------------------------
# Pin 5: uniform Abelian field -- closed form for the clover leaves, the 1/8 and the trace removal
# ---------------------------------------------------------------------------------------------
def abelian_links(dims, T, k=1):
    lx, ly, lz, lt = dims
    B = 2 * np.pi * k / (lx * ly)
    U = inputs.links_unit(dims).numpy()
    T = np.asarray(T, dtype=float)
    for xx in range(lx):
        U[:, :, :, xx, 1] = np.diag(np.exp(1j * B * xx * T))
    for yy in range(ly):
        U[:, :, yy, lx - 1, 0] = np.diag(np.exp(-1j * B * lx * yy * T))
    return U, B


def test_uniform_abelian_field_strength_closed_form():
    dims = (6, 4, 2, 2)
    U, B = abelian_links(dims, [1, -1, 0])
    F = oracle.field_strength(dims, U)
    expect = np.zeros_like(F)
    expect[..., 0, :, :] = np.sin(B) * np.diag([1.0, -1.0, 0.0])   # plane (x,y) only, at EVERY site
    assert np.abs(F - expect).max() < 1e-15
    # trace removal: T = diag(1,1,-2) -> sin(B T) - tr/3
    U, B = abelian_links(dims, [1, 1, -2])
    s = np.sin(B * np.array([1.0, 1.0, -2.0]))
    F = oracle.field_strength(dims, U, trace_sub=True)
    assert np.abs(F[..., 0, :, :] - np.diag(s - s.sum() / 3)).max() < 1e-15
    F = oracle.field_strength(dims, U, trace_sub=False)
    assert np.abs(F[..., 0, :, :] - np.diag(s)).max() < 1e-15
    # the clover block: A = 1 - kappa*csw*sigma_xy (x) F_xy with sigma_xy = diag(-1,+1,-1,+1)
    kappa, csw = 0.11, 0.9
    A = oracle.clover(dims, U, kappa, csw)
    sig_xy = np.diag([-1.0, 1.0, -1.0, 1.0])
    expect = np.eye(12) - kappa * csw * np.kron(sig_xy, np.diag(s - s.sum() / 3))
    assert np.abs(A - expect).max() < 1e-15


# ---------------------------------------------------------------------------------------------
# Pin 6: sign of the clover term relative to the Wilson term (zero-mode shift cancels at csw = 1)
# ---------------------------------------------------------------------------------------------
def _lowest_real_eig(dims, bc, U, kappa, csw):
    V = inputs.volume(dims)
    A = oracle.clover(dims, U, kappa, csw)
    n = 12 * V
    M = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    shape = (dims[3], dims[2], dims[1], dims[0], 4, 3)
    for k in range(n):
        e[k] = 1.0
        M[:, k] = oracle.M(dims, bc, U, A, kappa, e.reshape(shape)).ravel()
        e[k] = 0.0
    lam = np.linalg.eigvals(M)
    real = lam[np.abs(lam.imag) < 1e-9].real
    return real.min()


def test_clover_sign_zero_mode_shift():
    dims, bc, kappa = (6, 6, 2, 2), (1, 1, 1, 1), 0.11
    U, B = abelian_links(dims, [1, 1, -2])
    free = 1 - 8 * kappa
    shift = {c: (_lowest_real_eig(dims, bc, U, kappa, c) - free) / (kappa * B) for c in (0.0, 1.0, -1.0)}
    # SURVEY pin 6 (continuum algebra: D_W + clover = g.D - (g.D)^2/2 + (1-csw)/2 sigma.F):
    assert shift[0.0] > 0.5
    assert abs(shift[1.0]) < 0.1 * shift[0.0]
    assert shift[-1.0] > 1.8 * shift[0.0]


# ---------------------------------------------------------------------------------------------
# Pin 7: dense brute force on 2^4 and on a lattice with mixed extent-2 directions
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 4)])
def test_dense_bruteforce_matches_stencil(dims):
    kappa, csw = 0.12, 1.0
    U = np_links("haar", dims, seed=41)
    V = inputs.volume(dims)
    Md = bf.dense_M(dims, BC, U, kappa, csw)
    A = oracle.clover(dims, U, kappa, csw)
    assert rel(A, bf.clover_blocks(U, kappa, csw)) < 1e-14
    Ainv = oracle.clover_inverse(A)
    assert np.abs(A @ Ainv - np.eye(12)).max() < 1e-13
    shape = (dims[3], dims[2], dims[1], dims[0], 4, 3)
    n = 12 * V
    rng = np.random.default_rng(5)
    cols = range(n) if n <= 192 else rng.choice(n, 64, replace=False)
    e = np.zeros(n, dtype=np.complex128)
    for k in cols:
        e[k] = 1.0
        col = oracle.M(dims, BC, U, A, kappa, e.reshape(shape)).ravel()
        assert np.abs(col - Md[:, k]).max() < 1e-14
        cold = oracle.M(dims, BC, U, A, kappa, e.reshape(shape), dagger=True).ravel()
        assert np.abs(cold - Md.conj().T[:, k]).max() < 1e-14
        e[k] = 0.0
    # Schur complement from the dense matrix vs the oracle's masked composition
    Sd, ev, od = bf.dense_schur(dims, Md)
    x = rand_spinor(dims, 43) * (oracle.parity_mask(dims) == 0)[..., None, None]
    got = oracle.schur(dims, BC, U, A, Ainv, kappa, x).ravel()
    assert np.abs(got[od]).max() == 0
    assert rel(got[ev], Sd @ x.ravel()[ev]) < 1e-13
    gotd = oracle.schur(dims, BC, U, A, Ainv, kappa, x, dagger=True).ravel()
    assert rel(gotd[ev], Sd.conj().T @ x.ravel()[ev]) < 1e-13
    # parity dslash pieces: -kappa*D_eo is the even-odd block of M
    y = rand_spinor(dims, 44)
    d_eo = oracle.dslash_parity(dims, BC, U, 0, y).ravel()
    assert rel(-kappa * d_eo[ev], Md[np.ix_(ev, od)] @ y.ravel()[od]) < 1e-13
    d_oe = oracle.dslash_parity(dims, BC, U, 1, y).ravel()
    assert rel(-kappa * d_oe[od], Md[np.ix_(od, ev)] @ y.ravel()[ev]) < 1e-13


def test_dense_inverse_vs_cgnr_on_2to4():
    dims, kappa, csw = (2, 2, 2, 2), 0.12, 1.0
    U = np_links("haar", dims, seed=51)
    Md = bf.dense_M(dims, BC, U, kappa, csw)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 52)
    x_exact = np.linalg.solve(Md, b.ravel())
    for eo in (False, True):
        res = oracle.cgnr(dims, BC, U, A, Ainv, kappa, b, even_odd=eo, tol=1e-10)
        assert res["converged"]
        assert res["true_residual"] <= 1.05e-10
        assert rel(res["x"].ravel(), x_exact) < 5e-9
    # the oracle's own generic inverse against numpy's
    assert rel(oracle.dense_inverse(Md), np.linalg.inv(Md)) < 1e-10


# ---------------------------------------------------------------------------------------------
# Pins 8, 11: Schur identity, even-odd source preparation / reconstruction, monotone CGLS residual
# ---------------------------------------------------------------------------------------------
def test_schur_identity_and_monotone_residual():
    dims, kappa, csw = (4, 4, 4, 8), 0.1245, 1.0
    U = np_links("smooth", dims, seed=61)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 62)
    full = oracle.cgnr(dims, BC, U, A, Ainv, kappa, b, even_odd=False)
    eo = oracle.cgnr(dims, BC, U, A, Ainv, kappa, b, even_odd=True)
    assert full["converged"] and eo["converged"]
    assert full["true_residual"] <= 1.05e-10 and eo["true_residual"] <= 1.05e-10
    assert rel(eo["x"], full["x"]) < 2e-9
    assert eo["iters"] < full["iters"]          # even-odd preconditioning helps
    for h in (full["history"], eo["history"]):
        assert np.all(np.diff(h) <= 1e-14)      # CGNR minimises |b - Kx| over the Krylov space
    # block elimination written out: M [x_e; x_o] = b  <=>  S x_e = bhat_e, x_o = A_oo^-1(b_o + k D_oe x_e)
    mask_e = (oracle.parity_mask(dims) == 0)[..., None, None]
    x = full["x"]
    bhat = oracle.eo_prepare(dims, BC, U, Ainv, kappa, b)
    assert rel(oracle.schur(dims, BC, U, A, Ainv, kappa, x * mask_e), bhat) < 1e-9
    xr = oracle.eo_reconstruct(dims, BC, U, Ainv, kappa, b, x * mask_e)
    assert rel(xr, x) < 1e-9


def test_mixed_precision_model_matches_fp64_iteration_count():
    dims, kappa, csw = (4, 4, 4, 8), 0.1245, 1.0
    U = np_links("smooth", dims, seed=61)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 62)
    ref = oracle.cgnr(dims, BC, U, A, Ainv, kappa, b, even_odd=True)
    mix = oracle.cgnr_mixed(dims, BC, U, A, Ainv, kappa, b, even_odd=True, delta=0.1)
    assert mix["converged"] and mix["true_residual"] <= 1.05e-10
    assert mix["updates"] >= 2
    assert abs(mix["iters"] - ref["iters"]) <= max(1, int(np.ceil(0.02 * ref["iters"])))
    assert rel(mix["x"], ref["x"]) < 5e-9


@pytest.mark.parametrize("dims,even_odd", [((4, 4, 4, 8), True), ((4, 4, 4, 8), False), ((8, 8, 8, 16), True)])
@pytest.mark.parametrize("delta", [0.1, 0.01])
def test_reliable_update_schedule_is_pinned_by_the_fp64_history(dims, even_odd, delta):
    """SURVEY O8's schedule (rmax tracking, the delta test, when updates fire) pinned by something other than
    oracle_cgnr_mixed itself: the firing iterations follow from oracle_cgnr's fp64 residual history alone
    (tests/schedule.py), because the float-rounded recurrence tracks it to ~1e-6.  A mistake in the model -- rmax never
    reset, reset to the wrong value, delta off by a factor, <= for <, the update placed before the residual test --
    moves at least one firing iteration."""
    from schedule import reliable_update_schedule

    kappa, csw, tol = 0.1245, 1.0, 1e-10
    U = np_links("smooth", dims, seed=61)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 62)
    ref = oracle.cgnr(dims, BC, U, A, Ainv, kappa, b, even_odd=even_odd, tol=tol)
    mix = oracle.cgnr_mixed(dims, BC, U, A, Ainv, kappa, b, even_odd=even_odd, tol=tol, delta=delta)
    assert ref["converged"] and mix["converged"]
    rhs = oracle.eo_prepare(dims, BC, U, Ainv, kappa, b) if even_odd else b
    rmax0 = np.linalg.norm(rhs.ravel()) / np.linalg.norm(b.ravel())
    want, margin = reliable_update_schedule(ref["history"], rmax0, delta, tol)
    assert margin > 1e-4, "a delta decision sits on its threshold: pick another seed"
    # the float-rounded recurrence follows the fp64 one closely enough for the rule to be decided identically
    n = min(len(mix["history"]), len(ref["history"]))
    dev = np.abs(mix["history"][:n] - ref["history"][:n]) / ref["history"][:n]
    # Schur system: eps_fp32 * cond / delta ~ 6e-8 * 30 / 0.01 stays below 1e-4.  Unpreconditioned M: the rounded
    # recurrence loses conjugacy and LAGS the fp64 one; the bound is "by less than one pass", i.e. the deviation is
    # below the largest residual reduction of a single fp64 pass
    h = np.asarray(ref["history"])
    one_pass = float(np.max(1.0 - h[1:] / h[:-1]))
    assert dev.max() < (1e-4 if even_odd else one_pass), (float(dev.max()), one_pass)
    own, own_margin = reliable_update_schedule(mix["history"], rmax0, delta, tol)
    if even_odd:
        # well-conditioned Schur system: the recurrences agree to ~1e-6, so the fp64 history alone fixes the schedule
        assert mix["update_iters"] == want, (mix["update_iters"], want)
        assert mix["updates"] == len(want) and mix["iters"] == want[-1] == ref["iters"]
    else:
        # unpreconditioned M: the float-rounded recurrence drifts by per cent in the last decades, so a firing may move
        # by one pass against the fp64 prediction; the count may not
        assert len(mix["update_iters"]) == len(want)
        assert max(abs(a - b) for a, b in zip(mix["update_iters"], want)) <= 1, (mix["update_iters"], want)
    # the rule re-applied (here, in Python) to the recurrence's recorded history reproduces the firings exactly
    assert own_margin > 1e-6 and own == mix["update_iters"], (own, mix["update_iters"])
    # delta = 0.1 fires about once per decade, delta = 0.01 once per two decades
    decades = -np.log10(tol)
    assert abs(len(want) - decades / -np.log10(delta)) <= 2


# ---------------------------------------------------------------------------------------------
# Pin 9: clover block invariants
# ---------------------------------------------------------------------------------------------
def test_clover_block_invariants():
    dims, kappa, csw = (4, 4, 4, 4), 0.125, 1.2
    U = np_links("smooth", dims, seed=71, eps=0.4)
    A = oracle.clover(dims, U, kappa, csw)
    assert np.abs(A - bf.dag(A)).max() < 1e-15
    assert np.abs(A[..., :6, 6:]).max() == 0 and np.abs(A[..., 6:, :6]).max() == 0
    tr_up = np.einsum("...ii->...", A[..., :6, :6])
    tr_lo = np.einsum("...ii->...", A[..., 6:, 6:])
    assert np.abs(tr_up - 6).max() < 1e-14 and np.abs(tr_lo - 6).max() < 1e-14
    Ainv = oracle.clover_inverse(A)
    assert np.abs(Ainv @ A - np.eye(12)).max() < 1e-13
    ev = np.linalg.eigvalsh(A.reshape(-1, 12, 12))
    assert ev.min() > 0.5 and ev.max() < 1.5     # safely non-singular
    F = oracle.field_strength(dims, U)
    assert np.abs(F - bf.dag(F)).max() < 1e-15
    assert np.abs(np.einsum("...ii->...", F)).max() < 1e-15


# ---------------------------------------------------------------------------------------------
# O-L: sampled-site evaluation agrees with the full-lattice operators
# ---------------------------------------------------------------------------------------------
def test_apply_sites_matches_full_operators():
    dims, kappa, csw = (4, 6, 2, 4), 0.1245, 1.0
    U = np_links("smooth", dims, seed=81)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    psi = rand_spinor(dims, 82)
    V = inputs.volume(dims)
    sites = np.arange(V)
    full = {
        "D": oracle.hop(dims, BC, U, psi),
        "M": oracle.M(dims, BC, U, A, kappa, psi),
        "Mdag": oracle.M(dims, BC, U, A, kappa, psi, dagger=True),
    }
    for which, ref in full.items():
        got = oracle.apply_sites(dims, BC, U, kappa, csw, which, psi, sites)
        assert rel(got, ref.reshape(V, 4, 3)) < 1e-14
    mask_e = (oracle.parity_mask(dims) == 0)[..., None, None]
    for which, dg in (("S", False), ("Sdag", True)):
        ref = oracle.schur(dims, BC, U, A, Ainv, kappa, psi * mask_e, dagger=dg)
        got = oracle.apply_sites(dims, BC, U, kappa, csw, which, psi, sites)   # odd part of psi is ignored
        assert rel(got, ref.reshape(V, 4, 3)) < 1e-13


# ---------------------------------------------------------------------------------------------
# BiCGStab: pinned by the dense inverse, by CGNR's solution and by scipy's implementation
# ---------------------------------------------------------------------------------------------
def test_bicgstab_against_dense_inverse_and_cgnr():
    dims, kappa, csw = (2, 2, 2, 2), 0.12, 1.0
    U = np_links("haar", dims, seed=51)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    Md = bf.dense_M(dims, BC, U, kappa, csw)
    b = rand_spinor(dims, 52)
    x_exact = np.linalg.solve(Md, b.ravel())
    for eo in (False, True):
        res = oracle.bicgstab(dims, BC, U, A, Ainv, kappa, b, even_odd=eo)
        assert res["converged"] and not res["breakdown"]
        assert res["true_residual"] <= 1.05e-10
        assert rel(res["x"].ravel(), x_exact) < 5e-9
    dims = (4, 4, 4, 8)
    U = np_links("smooth", dims, seed=61)
    A = oracle.clover(dims, U, 0.1245, 1.0)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 62)
    cg = oracle.cgnr(dims, BC, U, A, Ainv, 0.1245, b, even_odd=True)
    for eo in (False, True):
        bi = oracle.bicgstab(dims, BC, U, A, Ainv, 0.1245, b, even_odd=eo)
        assert bi["converged"] and bi["true_residual"] <= 1.05e-10
        assert rel(bi["x"], cg["x"]) < 5e-9
    # half the operator applications per pass of CGNR's, and fewer passes: the point of the method
    assert bi["iters"] < cg["iters"]


def test_bicgstab_iterates_match_scipy():
    """The same recurrence in a library: scipy.sparse.linalg.bicgstab on a LinearOperator that applies the oracle's Schur
    operator, x0 = 0, no preconditioner.  Iterate by iterate (scipy's callback) the two agree to rounding until rounding
    differences have been amplified (late in the solve); a wrong coefficient, a swapped conjugation in <t, s> or a
    wrong update order shows in the first iterate."""
    from scipy.sparse.linalg import LinearOperator, bicgstab as sp_bicgstab

    dims, kappa, csw = (4, 4, 4, 4), 0.124, 1.0
    U = np_links("smooth", dims, seed=91)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    b = rand_spinor(dims, 92)
    mask_e = (oracle.parity_mask(dims) == 0)[..., None, None]
    shape = b.shape
    idx = np.flatnonzero(np.broadcast_to(mask_e, shape).ravel())

    def S(xe):
        full = np.zeros(b.size, dtype=np.complex128)
        full[idx] = xe
        return oracle.schur(dims, BC, U, A, Ainv, kappa, full.reshape(shape)).ravel()[idx]

    n = idx.size
    op = LinearOperator((n, n), matvec=S, dtype=np.complex128)
    bhat = oracle.eo_prepare(dims, BC, U, Ainv, kappa, b).ravel()[idx]
    iterates = []
    x_sp, info = sp_bicgstab(op, bhat, x0=np.zeros(n, dtype=np.complex128), rtol=1e-12, atol=0.0, maxiter=12,
                             callback=lambda xk: iterates.append(xk.copy()))
    assert len(iterates) >= 8
    bnorm = np.linalg.norm(b.ravel())
    for k, xk in enumerate(iterates[:8]):
        ours = oracle.bicgstab(dims, BC, U, A, Ainv, kappa, b, even_odd=True, tol=1e-30, max_iter=k + 1)
        xe = ours["x"].ravel()[idx]          # even part of the reconstructed solution = the Schur iterate
        assert rel(xe, xk) < 1e-9, (k, rel(xe, xk))
        # and the recorded residual is the residual of that iterate
        assert abs(ours["history"][k] - np.linalg.norm(bhat - S(xk)) / bnorm) <= 1e-9 * ours["history"][0]


# ---------------------------------------------------------------------------------------------
# Low modes of S^+ S: pinned by the brute-force dense matrix
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 4)])
def test_lowest_modes_against_brute_force_dense_schur(dims):
    """oracle.lowest_modes against the Schur complement of the independent numpy brute-force matrix (tests/bruteforce.py:
    hand-typed gammas, np.roll clover), both through its dense path and through its ARPACK path."""
    kappa, csw = 0.124, 1.0
    U = np_links("smooth", dims, seed=95)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    Md = bf.dense_M(dims, BC, U, kappa, csw)
    par = np.repeat(oracle.parity_mask(dims).ravel(), 12)
    e, o = np.flatnonzero(par == 0), np.flatnonzero(par == 1)
    Sd = Md[np.ix_(e, e)] - Md[np.ix_(e, o)] @ np.linalg.solve(Md[np.ix_(o, o)], Md[np.ix_(o, e)])
    want = np.linalg.eigvalsh(Sd.conj().T @ Sd)
    k = 6
    w, v = oracle.lowest_modes(dims, BC, U, A, Ainv, kappa, k)
    assert np.allclose(w, want[:k], rtol=1e-10, atol=0)
    assert w[0] > 0 and np.all(np.diff(w) >= 0)
    # eigenvector property with the oracle's own operator, orthonormality, support on the even sites only
    for i in range(k):
        Hv = oracle.schur(dims, BC, U, A, Ainv, kappa, oracle.schur(dims, BC, U, A, Ainv, kappa, v[i]), dagger=True)
        assert np.linalg.norm((Hv - w[i] * v[i]).ravel()) < 1e-10
        assert abs(np.linalg.norm(v[i].ravel()) - 1) < 1e-12
        assert np.abs(v[i][oracle.parity_mask(dims) == 1]).max() == 0
    w2, v2 = oracle.lowest_modes(dims, BC, U, A, Ainv, kappa, k, dense_limit=0)
    assert np.allclose(w2, want[:k], rtol=1e-9, atol=0)
