"""qxd_norm2_noalloc (include/qxd.h, csrc/noalloc.cu): the allocation-free variant of the norm reduction against the
existing path (qxd_blas_norm2_dev, partial sums in the caller's workspace) on the same packed spinors.

Collected last on purpose (file name): the suite runs with ``pytest -x``.  Works alone in a fresh process and after the
other tests: it builds its own context and depends on nothing they leave behind.
"""
import ctypes as C

import numpy as np
import pytest

import synth

F64, F32 = 0, 1


def _packed_norms(g, B, torch, eta, prec):
    """(existing path, new entry point) for the even half of the packed spinor; the new one twice in a row on the same input."""
    packed = g.spinor_pack(eta, prec)
    hb = g.packed_spinor_bytes(prec, half_only=True)
    half = packed[:hb]
    ref = torch.zeros(1, dtype=torch.float64, device="cuda")
    g.blas_norm2_dev(half, prec, ref)
    flat = half.view(torch.float64 if prec == F64 else torch.float32)
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    B.norm2_noalloc(flat, out[0:1])
    B.norm2_noalloc(flat, out[1:2])
    torch.cuda.synchronize()
    return float(ref[0]), out.cpu().numpy(), flat


@pytest.mark.gpu
@pytest.mark.parametrize("dims,cstar", [((8, 8, 8, 8), 0), ((12, 6, 4, 10), 3)])
def test_norm2_noalloc_matches_workspace_path(dims, cstar):
    import torch
    from paper_2502_02490_b200 import binding as B
    bc = cstar | (1 << 2)
    g = B.Qxd(*dims, bc, precisions=(F64, F32))
    dims_ext = (dims[0], 2 * dims[1] if cstar else dims[1], dims[2], dims[3])
    eta = torch.from_numpy(synth.gaussian_spinor(dims_ext, 3)).cuda()
    for prec, tol in ((F64, 1e-13), (F32, 1e-6)):       # north_star's tolerances for fp64 / fp32 (tests/test_gpu_parity.py)
        ref, got, flat = _packed_norms(g, B, torch, eta, prec)
        assert ref > 0.0
        assert abs(got[0] - ref) <= tol * ref, (prec, got, ref)
        assert got[1] == got[0], "two calls in a row on the same input must agree bit for bit (fixed chunks, fixed order)"
        # and against plain arithmetic on the same numbers
        plain = float((flat.double() ** 2).sum())
        assert abs(got[0] - plain) <= 1e-13 * plain
    # a second, DIFFERENT and shorter input right after a longer one: stale partial sums of the previous call must not leak
    short = flat[: 4096 + 37].contiguous()
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    B.norm2_noalloc(short, out)
    assert abs(float(out[0]) - float((short.double() ** 2).sum())) <= 1e-13 * float(out[0])
    z = torch.empty(0, dtype=torch.float64, device="cuda")
    B.norm2_noalloc(z, out)
    assert float(out[0]) == 0.0
    g.close()


@pytest.mark.gpu
def test_norm2_noalloc_allocates_nothing_and_rejects_oversize():
    import torch
    from paper_2502_02490_b200 import binding as B
    lib = B.load_library()
    assert lib.qxd_noalloc_init() == 0
    x = torch.from_numpy(np.random.default_rng(5).normal(size=3 * 4096 + 5)).cuda()
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    B.norm2_noalloc(x, out)                      # warm: module loaded, set-up done
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        B.norm2_noalloc(x, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "the entry point must not allocate device memory"
    assert abs(float(out[0]) - float((x ** 2).sum())) <= 1e-13 * float(out[0])
    # beyond the static scratch: rejected before anything is launched (the pointer is never dereferenced)
    nmax = B.noalloc_max_reals()
    assert nmax == 65536 * 4096
    rc = lib.qxd_norm2_noalloc(F64, C.c_void_p(x.data_ptr()), nmax + 1, C.c_void_p(out.data_ptr()), None)
    assert rc == B.QXD_EINVAL
    msg = lib.qxd_noalloc_last_error().decode()
    assert "exceed" in msg and str(nmax) in msg
    assert lib.qxd_norm2_noalloc(2, C.c_void_p(x.data_ptr()), 16, C.c_void_p(out.data_ptr()), None) == B.QXD_EINVAL     # fp16: not a flat array
    assert lib.qxd_norm2_noalloc(F64, None, 16, C.c_void_p(out.data_ptr()), None) == B.QXD_EINVAL
