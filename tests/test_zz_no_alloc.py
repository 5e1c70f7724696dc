"""gd_energy_static -- the energy call for programs that cannot allocate GPU memory.

Everything else in the library runs out of a workspace that the caller obtained from cudaMalloc, and gd_init pins host
memory on top.  That is not possible everywhere: a driver that handed all free HBM to its own pool at start-up gets
"out of memory" from any later cudaMalloc, a time-critical loop cannot take the device-wide wait that cudaMalloc and
cudaFree cause, and a plug-in may sit inside an application that forbids allocations once it runs.  gd_energy_static
serves those callers: its only scratch is a fixed array built into the library (128 KiB on each GPU, good for up to
GD_ENERGY_STATIC_MAX_N = 2^21 particles), and the caller passes nothing but its own input and output buffers.

The tests here hold the new call to the existing one (gd_init + gd_energy, which is itself held to the oracle in
test_gpu_parity.py) at the tolerance the energy tests use, 1e-13 relative, on calls made back to back -- the built-in
array is shared by all calls and keeps the previous call's numbers, so the second and third results must not depend
on what the first left behind -- and check that a second call leaves the GPU's free memory untouched.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide another
test.  It passes on its own in a fresh process and at the end of the whole suite.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1702_00440_b200 import workloads as W

TOL = 1e-13          # relative, as test_gpu_parity.py::test_energy_matches_oracle


def test_static_energy_refuses_sizes_beyond_its_array_without_a_gpu():
    # argument checks run before the first CUDA call, so this needs no device: pointers are never dereferenced
    from paper_1702_00440_b200 import binding, build
    build.build_library()
    lib = binding.load()
    limit = binding.ENERGY_STATIC_MAX_N
    header = (build.INCLUDE / "gravidy_b200.h").read_text()
    assert f"#define GD_ENERGY_STATIC_MAX_N {limit}" in header
    assert lib.gd_energy_static(limit + 1, 256, 256, 256, 1e-4, 256, None) == binding.GD_EINVAL
    text = lib.gd_energy_static_last_error().decode()
    assert str(limit) in text and str(limit + 1) in text and "gd_energy_static" in text
    assert lib.gd_energy_static(0, 256, 256, 256, 1e-4, 256, None) == binding.GD_EINVAL
    assert lib.gd_energy_static(16, None, 256, 256, 1e-4, 256, None) == binding.GD_EINVAL
    assert lib.gd_energy_static(16, 256, 256, 256, 1e-4, None, None) == binding.GD_EINVAL
    assert lib.gd_energy_static(16, 256, 256, 256, -1.0, 256, None) == binding.GD_EINVAL
    assert lib.gd_energy_static(16, 256, 256, 256, float("nan"), 256, None) == binding.GD_EINVAL
    assert b"eps" in lib.gd_energy_static_last_error()


@pytest.fixture(scope="module")
def gd():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (the product has no CPU fallback)")
    from paper_1702_00440_b200 import binding
    binding.load()
    return binding


def existing_path(gd, w):
    """K, U from the call the library already had: a context on a cudaMalloc'ed workspace, then gd_energy."""
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    K, U = h.energy()
    h.close()
    return K, U


@pytest.mark.gpu
def test_static_energy_matches_the_workspace_path_on_calls_in_a_row(gd):
    import torch
    # a long system first (24 tiles, ragged tail), then a short one (6 tiles, ragged): the second call finds the first
    # call's 24 partial sums in the shared array and must use only the 6 it writes itself; then the long one again
    big, small = W.config(4, n=6001), W.config(1, n=1300)
    expect = {id(w): existing_path(gd, w) for w in (big, small)}
    dev = {id(w): [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.m, w.x, w.v)] for w in (big, small)}
    outs = [torch.full((2,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    torch.cuda.synchronize()

    # the very first call on this GPU does the one-time address look-up; the calls after it are the steady state
    gd.energy_static(*dev[id(big)], big.eps, outs[0])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    gd.energy_static(*dev[id(small)], small.eps, outs[1])          # two calls in a row, nothing in between
    gd.energy_static(*dev[id(big)], big.eps, outs[2])
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]

    for w, out in ((big, outs[0]), (small, outs[1]), (big, outs[2])):
        K, U = out.cpu().numpy()
        K_ref, U_ref = expect[id(w)]
        assert abs(K / K_ref - 1) < TOL and abs(U / U_ref - 1) < TOL, (w.m.shape[0], K, K_ref, U, U_ref)
    # same input, same bits, whatever the array held before
    assert np.array_equal(outs[0].cpu().numpy(), outs[2].cpu().numpy())
    # nothing was taken from (or given back to) the device by the steady-state calls
    assert free_after == free_before


@pytest.mark.gpu
def test_static_energy_edge_sizes_and_a_side_stream(gd):
    import torch
    s = torch.cuda.Stream()
    for n, eps in ((1, 1e-4), (2, 0.0), (256, 1e-4), (257, 0.0)):
        w = W.random_cluster(n, seed=900 + n, eps=eps)
        K_ref, U_ref = existing_path(gd, w)
        m, x, v = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.m, w.x, w.v))
        out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        gd.energy_static(m, x, v, eps, out, stream=s)
        s.synchronize()
        K, U = out.cpu().numpy()
        assert abs(K - K_ref) <= TOL * abs(K_ref) and abs(U - U_ref) <= TOL * abs(U_ref), (n, K, K_ref, U, U_ref)
    # the binding refuses to convert (= allocate) on the caller's behalf
    with pytest.raises(AssertionError):
        gd.energy_static(m.float(), x, v, eps, out)
    # and the size limit is enforced with a GPU present as well
    rc = gd.load().gd_energy_static(gd.ENERGY_STATIC_MAX_N + 1, m.data_ptr(), x.data_ptr(), v.data_ptr(), 1e-4,
                                    out.data_ptr(), None)
    assert rc == gd.GD_EINVAL and b"GD_ENERGY_STATIC_MAX_N" in gd.load().gd_energy_static_last_error()
