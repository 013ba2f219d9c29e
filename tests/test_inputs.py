"""Seeded input generators (paper_2302_00850_b200/inputs.py): hash pinned to the published splitmix64
outputs, SU(3) properties of the links (SURVEY.md §8(d), §8(c) pin 10), reproducibility.  CPU only."""
import os

import numpy as np
import torch

from paper_2302_00850_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "splitmix64.txt")


def test_splitmix64_matches_published_vectors():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 2
    for xin, xout in rows:
        x, want = int(xin, 16), int(xout, 16)
        assert inputs.splitmix64_int(x) == want
        got = inputs.splitmix64(torch.tensor([inputs._i64(x)], dtype=torch.int64)).item() & ((1 << 64) - 1)
        assert got == want


def test_tensor_hash_equals_scalar_hash_on_random_words():
    rng = np.random.default_rng(0)
    xs = [int(v) for v in rng.integers(0, 2**63, size=64)] + [2**64 - 1, 2**63, 2**63 + 12345]
    t = torch.tensor([inputs._i64(x) for x in xs], dtype=torch.int64)
    got = [int(v) & ((1 << 64) - 1) for v in inputs.splitmix64(t).tolist()]
    assert got == [inputs.splitmix64_int(x) for x in xs]


def test_normals_are_counter_based_and_standard():
    idx = torch.arange(200000, dtype=torch.int64)
    a = inputs.normals(5, inputs.STREAM_SOURCE, idx, 4)
    b = inputs.normals(5, inputs.STREAM_SOURCE, idx[1000:1010], 4)
    assert torch.equal(a[1000:1010], b)                       # value depends on the index only
    assert not torch.equal(a, inputs.normals(6, inputs.STREAM_SOURCE, idx, 4))
    assert not torch.equal(a, inputs.normals(5, inputs.STREAM_LINKS, idx, 4))
    assert abs(a.mean().item()) < 5e-3 and abs(a.var().item() - 1.0) < 1e-2
    assert abs((a ** 4).mean().item() - 3.0) < 0.05


def _check_su3(u):
    u = u.reshape(-1, 3, 3)
    eye = torch.eye(3, dtype=u.dtype)
    assert (u @ u.conj().transpose(-1, -2) - eye).abs().max().item() < 1e-14
    assert (torch.linalg.det(u) - 1).abs().max().item() < 1e-13
    # SURVEY pin 10: third row = conj(row1 x row2) (what 12-real compression relies on)
    r3 = torch.linalg.cross(u[:, 0], u[:, 1]).conj()
    assert (r3 - u[:, 2]).abs().max().item() < 1e-14


def test_links_are_su3_with_expected_plaquette():
    dims = (4, 4, 4, 8)
    haar = inputs.links_haar(dims, 3)
    smooth = inputs.links_smooth(dims, 0.3, 3)
    _check_su3(haar)
    _check_su3(smooth)
    assert abs(inputs.plaquette(haar)) < 0.05                  # plaquette ~ 0
    assert abs(inputs.plaquette(smooth) - 0.785) < 0.01        # plaquette ~ 0.785
    assert abs(inputs.plaquette(inputs.links_smooth(dims, 0.4, 3)) - 0.646) < 0.015
    assert inputs.plaquette(inputs.links_unit(dims)) == 1.0
    # chunked generation is layout independent
    assert torch.equal(smooth, inputs.links_smooth(dims, 0.3, 3, chunk=1000))


def test_gauge_transformed_links_stay_su3_and_sources_are_well_formed():
    dims = (4, 2, 4, 4)
    u = inputs.links_haar(dims, 9)
    g = inputs.su3_site_field(dims, 10)
    _check_su3(g)
    _check_su3(inputs.gauge_transform_links(u, g))
    s = inputs.source_smeared(dims, inputs.links_smooth(dims, 0.3, 9))
    assert abs(torch.linalg.vector_norm(s).item() - 1) < 1e-14
    assert s[1:].abs().max().item() == 0                        # smearing stays on time-slice 0
    assert s[0][..., 0, :].abs().min().item() > 0 and s[0][..., 1:, :].abs().max().item() == 0
    p = inputs.source_point(dims, 2, 1)
    assert p.abs().sum().item() == 1 and p[0, 0, 0, 0, 2, 1] == 1
    for k, c in inputs.CONFIGS.items():
        assert all(e % 2 == 0 for e in c["dims"])
