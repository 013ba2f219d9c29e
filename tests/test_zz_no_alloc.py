"""cola_spinor_norm2_static -- the entry point for callers that may not allocate GPU memory.

Every other call of the library needs a context (cola_create allocates a small control block and pinned host memory)
and a workspace that somebody allocated and lent to it.  A caller that was only handed device pointers -- a hook running
after the host application's memory pool has taken the whole GPU, or inside a loop where cudaMalloc's device-wide
synchronisation is not acceptable -- can use neither.  For it the library offers |v|^2 with the reduction's scratch in a
16 KB array inside the library's own device image (include/cola.h, csrc/cola_static.cu).

Checked here: the result against the regular path (cola_spinor_norm2, scratch in the lent workspace) within the
tolerances of the parity tests (1e-12 fp64, 2e-6 fp32; the two are in fact the same bits) on consecutive calls that
reuse the shared array without a synchronisation in between, with sizes that shrink from call to call so that stale
partials of the earlier call sit right behind the later call's; free device memory unchanged across calls; sizes
above the stated maximum and malformed arguments refused with a message.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this add-on must not hide
the parity tests.  It passes on its own in a fresh process and after the rest of the suite.
"""
import ctypes

import pytest
import torch

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-12, torch.float32: 2e-6}


@pytest.fixture(scope="module")
def binding():
    from paper_2302_00850_b200 import binding

    assert torch.cuda.is_available()
    return binding


def internal_vector(ctx, dtype, full, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    shape = ctx.empty_internal(dtype, full=full).shape
    return torch.randn(shape, dtype=torch.float64, generator=g).to(dtype).cuda()


def test_two_calls_in_a_row_match_the_workspace_path(binding):
    # (lattice, precision, full lattice?) in the order the static entry point is called: 1184 blocks (the grid cap, 5
    # reduction groups, grid-stride loop), then 384 blocks in 2 groups, then 34 blocks of a ragged half lattice.
    cases = [((16, 16, 16, 32), torch.float32, True), ((8, 8, 8, 16), torch.float64, True), ((12, 10, 6, 4), torch.float32, False)]
    ctxs, vecs, want = [], [], []
    for k, (dims, dtype, full) in enumerate(cases):
        c = binding.Cola(dims, 0.12, 1.0)
        c.set_workspace()
        v = internal_vector(c, dtype, full, seed=100 + k)
        want.append(c.spinor_norm2(v))          # regular path: scratch in the context's workspace
        ctxs.append(c)
        vecs.append(v)
    out = torch.full((len(cases),), -1.0, dtype=torch.float64, device="cuda")
    got = [binding.spinor_norm2_static(v, out=out[k:k + 1]) for k, v in enumerate(vecs)]   # back to back, one stream, no sync
    torch.cuda.synchronize()
    for (dims, dtype, full), v, g, w in zip(cases, vecs, got, want):
        g, w = g.item(), w.item()
        ref = (v.double() ** 2).sum().item()
        assert w > 0 and abs(g - w) <= TOL[dtype] * w, (dims, dtype, g, w)
        assert g == w, "same grid and summation order: expected identical bits"
        assert abs(g - ref) <= TOL[dtype] * ref, (dims, dtype, g, ref)
    # a second round in the opposite order gives the same numbers: nothing a call leaves in the shared array matters
    again = [binding.spinor_norm2_static(v).item() for v in reversed(vecs)]
    assert again == [g.item() for g in reversed(got)]
    for c in ctxs:
        c.close()


def test_calls_leave_free_device_memory_unchanged(binding):
    v = torch.randn(6, 4096, 4, dtype=torch.float32, device="cuda")
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    binding.spinor_norm2_static(v, out=out)     # first use on this device: address look-up (and module load)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        binding.spinor_norm2_static(v, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert abs(out.item() - (v.double() ** 2).sum().item()) <= 2e-6 * out.item()


def test_sizes_beyond_the_maximum_and_bad_arguments_are_refused(binding):
    lib = binding._lib
    v = torch.ones(6, 64, 4, dtype=torch.float32, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    vp, op = ctypes.c_void_p(v.data_ptr()), ctypes.c_void_p(out.data_ptr())

    def call(device=0, prec=binding.COLA_F32, vptr=vp, n=64, optr=op):
        st = lib.cola_spinor_norm2_static(device, None, prec, vptr, n, optr)
        return st, lib.cola_last_error(None).decode()

    st, msg = call(n=binding.COLA_STATIC_MAX_SITES + 1)     # rejected before the pointer is touched
    assert st == binding.COLA_EINVAL and "COLA_STATIC_MAX_SITES" in msg
    assert call(n=0)[0] == binding.COLA_EINVAL
    assert call(vptr=None)[0] == binding.COLA_EINVAL
    assert call(optr=None)[0] == binding.COLA_EINVAL
    assert call(prec=binding.COLA_F32_H16)[0] == binding.COLA_EINVAL
    assert call(device=-1)[0] == binding.COLA_EINVAL
    st, msg = call()
    torch.cuda.synchronize()
    assert st == binding.COLA_OK and out.item() == 64 * 24
