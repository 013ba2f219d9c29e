"""Writes tests/golden/solver_golden.json: iteration counts, residuals and sampled solution values of the
CPU oracle (oracle/ only -- no CUDA code is imported) for BASELINE.json configs 0, 1, 2.

    python tests/golden/make_golden.py [config ...]

The 32^3x64 solve (config 2) takes ~15-30 min on 8 cores, which is why its numbers are stored rather
than recomputed in the GPU tests.  Inputs come from paper_2302_00850_b200.inputs (seeded generators).
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2302_00850_b200 import inputs  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "solver_golden.json")
N_SAMPLE = 64


def sample_sites(volume, k):
    rng = np.random.default_rng(1000 + k)
    return np.sort(rng.choice(volume, size=min(N_SAMPLE, volume), replace=False))


def run(k):
    c = inputs.CONFIGS[k]
    dims = c["dims"]
    U = inputs.make_links(k)
    b = inputs.make_source(k, u=U).numpy()
    U = U.numpy()
    A = oracle.clover(dims, U, c["kappa"], c["csw"])
    Ainv = oracle.clover_inverse(A)
    entry = dict(dims=list(dims), kappa=c["kappa"], csw=c["csw"], threads=oracle.num_threads())
    modes = [("eo", True)] + ([("full", False)] if k == 0 else [])
    for name, eo in modes:
        t0 = time.time()
        r = oracle.cgnr(dims, inputs.BC, U, A, Ainv, c["kappa"], b, even_odd=eo, tol=1e-10)
        sites = sample_sites(inputs.volume(dims), k)
        # |r_0| / |b| of the iterated system and the residual history |r_{k+1}| / |b|: what the reliable-update schedule
        # of the mixed-precision solvers follows from (tests/schedule.py)
        rhs = oracle.eo_prepare(dims, inputs.BC, U, Ainv, c["kappa"], b) if eo else b
        rmax0 = float(np.linalg.norm(rhs.ravel()) / np.linalg.norm(b.ravel()))
        xs = r["x"].reshape(-1, 12)[sites]
        entry[name] = dict(iters=int(r["iters"]), converged=bool(r["converged"]), true_residual=float(r["true_residual"]),
                           x_norm=float(np.linalg.norm(r["x"].ravel())), sites=[int(s) for s in sites],
                           x_re=[[float(v) for v in row.real] for row in xs], x_im=[[float(v) for v in row.imag] for row in xs],
                           rmax0=rmax0, history=[float(v) for v in r["history"]],
                           seconds=time.time() - t0)
        print(k, name, entry[name]["iters"], entry[name]["true_residual"], entry[name]["seconds"], flush=True)
    return entry


if __name__ == "__main__":
    ks = [int(a) for a in sys.argv[1:]] or [0, 1, 2]
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for k in ks:
        data[str(k)] = run(k)
        json.dump(data, open(OUT, "w"), indent=1)
