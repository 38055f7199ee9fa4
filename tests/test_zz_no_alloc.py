"""ic_largest_cluster_static -- the one entry point of the library that needs no memory from its caller beyond input and output.

Who it is for: code that cannot allocate device memory at the moment it wants the size of the charge drop
(PAPER.md:161-163).  Examples: an analysis hook called inside another program's time step after that program has given all
of HBM to its own pool; a plug-in whose host forbids cudaMalloc / cudaFree while it runs because both wait for the whole
device and stall every other stream; a monitor with a fixed memory budget.  Every other call of the library takes a
caller-allocated workspace or scratch buffer; this one keeps its union-find arrays in an 8 MiB array that is part of the
library itself (one per GPU, shared by all calls, so L <= 1024 and no two calls may overlap on the GPU).

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  The GPU test passes on its own in a fresh process (the first call then does the per-device set-up) and
after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

import ic_inputs


def test_static_cluster_rejects_bad_arguments_before_touching_the_gpu():
    """Sizes beyond the built-in array get an error of their own, with a text that names the limit and the way out; the
    argument checks come before any CUDA call, so this runs without a GPU."""
    import paper_2301_11735_b200 as pkg
    f = pkg.lib.ic_largest_cluster_static
    p = C.c_void_p(4096)           # never dereferenced: every case below is rejected first
    assert f(None, 64, 0, p, None) == pkg.IC_ERR_NULL and f(p, 64, 0, None, None) == pkg.IC_ERR_NULL
    for L in (0, 2, 3, 48, -64):
        assert f(p, L, 0, p, None) == pkg.IC_ERR_SIZE, L
    for L in (2048, 4096, 1 << 20):
        assert f(p, L, 0, p, None) == pkg.IC_ERR_STATIC_MAX, L
    for which in (-1, 3):
        assert f(p, 64, which, p, None) == pkg.IC_ERR_PARAM
    text = pkg.lib.ic_strerror(pkg.IC_ERR_STATIC_MAX).decode()
    assert str(pkg.IC_STATIC_CLUSTER_MAX_L) in text and "ic_largest_cluster" in text
    assert pkg.IC_STATIC_CLUSTER_MAX_L == 1024


@pytest.mark.gpu
def test_static_cluster_equals_the_scratch_buffer_path_on_calls_in_a_row():
    """Calls in a row on the shared array give exactly what ic_largest_cluster gives with a caller-allocated scratch buffer
    (integers: equality, the tolerance of every cluster test here): the maximum size first, then a smaller lattice that
    leaves three quarters of the previous forest in the array, then the first lattice again with another selection, all near
    the site-percolation threshold where clusters are large and ragged.  The second and later calls leave the amount of free
    device memory unchanged."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2301_11735_b200 as pkg

    def lattice(L, dens, seed):
        N = L * L
        nplus, nminus = int(dens * N * 0.6), int(dens * N * 0.4)
        return ic_inputs.random_state(L, nplus, nminus, seed, 0), (nplus - nminus) / N

    want, dev = {}, {}
    for name, (L, dens, seed) in {"big": (1024, 0.59, 71), "mid": (256, 0.5, 72), "tiny": (4, 0.5, 73)}.items():
        code, n = lattice(L, dens, seed)
        sim = pkg.Sim(L, n, 0.5, 1.0, 1.0, seed=1)              # the existing path: context + workspace + scratch tensor
        sim.set_state(0, code)
        want[name] = [sim.largest_cluster(0, which) for which in (0, 1, 2)]
        sim.close()
        dev[name] = torch.from_numpy(np.ascontiguousarray(code, dtype=np.int8)).cuda()
    assert want["big"][0][0] > 1000 and want["big"][0][1] > 1000        # a real forest, not a trivial lattice
    out = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()

    def call(name, which):
        pkg.largest_cluster_static(dev[name], which, out)
        torch.cuda.synchronize()
        return tuple(int(v) for v in out.tolist())

    assert call("big", 0) == want["big"][0]                    # first call of the process on this device: does the set-up
    free_before = torch.cuda.mem_get_info()[0]
    assert call("big", 0) == want["big"][0]                    # the same again on the array the first call left behind
    assert call("mid", 1) == want["mid"][1]                    # smaller: most of the array still holds the big forest
    assert call("big", 2) == want["big"][2]
    assert call("tiny", 0) == want["tiny"][0]
    assert call("big", 1) == want["big"][1]
    assert torch.cuda.mem_get_info()[0] == free_before, "a call after the first changed the free device memory"

    # calls queued back to back on one stream, no host synchronisation in between: in-order execution is enough
    outs = [torch.empty(2, dtype=torch.int64, device="cuda") for _ in range(4)]
    order = [("mid", 0), ("big", 0), ("mid", 2), ("tiny", 1)]
    for o, (name, which) in zip(outs, order):
        pkg.largest_cluster_static(dev[name], which, o)
    torch.cuda.synchronize()
    assert [tuple(o.tolist()) for o in outs] == [want[name][which] for name, which in order]

    # a pointer the GPU cannot read (ordinary host memory) is refused instead of faulting in a kernel
    host = np.zeros((64, 64), dtype=np.int8)
    rc = pkg.lib.ic_largest_cluster_static(C.c_void_p(host.ctypes.data), 64, 0, C.c_void_p(out.data_ptr()), None)
    assert rc == pkg.IC_ERR_PARAM
    # too large for the built-in array: refused, the output untouched
    big = torch.zeros((2048, 2048), dtype=torch.int8, device="cuda")
    out.fill_(-7)
    with pytest.raises(pkg.IcError) as e:
        pkg.largest_cluster_static(big, 0, out)
    assert e.value.code == pkg.IC_ERR_STATIC_MAX
    torch.cuda.synchronize()
    assert out.tolist() == [-7, -7]
