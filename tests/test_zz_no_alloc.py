"""rbmf_prepare_strain_static: the front end for callers that cannot hand the library any device memory.

Every other entry point of librbmf.so works out of a caller-allocated workspace, and rbmf_prepare_strain needs a whole
plan to borrow three small scratch arrays from.  A whitening stage that owns no plan, a callback inside another
program's pipeline that only receives its input and output buffers, or a process whose memory pool has already taken the
whole GPU cannot provide that, so this one entry point keeps its scratch in a fixed 12 MiB array inside the library
(include/rbmf.h has the full contract: at most 2^20 samples per call, one shared array per GPU, calls must not overlap).

The file sorts last on purpose: the GPU test below must pass both alone in a fresh process and after every other test
has used the library (and left its own data in the GPU's memory), and a failure here cannot hide another file's tests
behind `pytest -x`.
"""
import ctypes

import numpy as np
import pytest


@pytest.fixture(scope="module")
def rbmf(built_library):
    from paper_2110_13115_b200 import rbmf as mod
    return mod


def test_static_limits_and_argument_checks(rbmf):
    """Host-side contract (no GPU needed): the stated maximum, and that anything beyond it is refused before a single
    CUDA call is made -- RBMF_ERR_UNSUPPORTED for a valid request that exceeds the fixed array, RBMF_ERR_ARG for a
    request no entry point would take."""
    b = rbmf
    max_samples, nbytes = ctypes.c_int64(), ctypes.c_size_t()
    assert b.rbmf_prepare_strain_static_limits(ctypes.byref(max_samples), ctypes.byref(nbytes)) == b.RBMF_OK
    assert max_samples.value == 1 << 20 and nbytes.value == 12 << 20
    assert b.rbmf_prepare_strain_static_limits(None, None) == b.RBMF_OK
    dummy, err = 1024, ctypes.c_int32(99)      # a non-NULL, 8-byte aligned address that is never dereferenced here
    for N, nb in ((1 << 21, 1), (1 << 24, 1), (1 << 20, 2), (1 << 19, 3), (1 << 10, 1025)):
        assert b.rbmf_prepare_strain_static(dummy, None, N, nb, dummy, None, ctypes.byref(err)) == b.RBMF_ERR_UNSUPPORTED
        assert err.value == 0
    for N, nb in ((1000, 1), (512, 1), (1 << 25, 1), (4096, 0), (4096, -1)):
        assert b.rbmf_prepare_strain_static(dummy, None, N, nb, dummy, None, None) == b.RBMF_ERR_ARG
    assert b.rbmf_prepare_strain_static(None, None, 4096, 1, dummy, None, None) == b.RBMF_ERR_ARG
    assert b.rbmf_prepare_strain_static(dummy, None, 4096, 1, None, None, None) == b.RBMF_ERR_ARG
    assert b.rbmf_prepare_strain_static(dummy + 4, None, 4096, 1, dummy, None, None) == b.RBMF_ERR_ARG


def _series(N, nb, seed):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((nb, N)).astype(np.float32)
    x[-1] += (3.0 * np.cos(2 * np.pi * 37 * np.arange(N) / N + 0.4)).astype(np.float32)
    inv_asd = rng.uniform(0.5, 2.0, N // 2 + 1).astype(np.float32)
    return x, inv_asd


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path(rbmf):
    """The no-allocation entry point against the existing one (rbmf_prepare_strain, scratch in the plan's workspace),
    on calls made back to back that share the fixed array: a batch of four short segments, then one segment of the
    largest size the array takes (2^20 samples, which overwrites all of it, twiddle table included), then the first
    input again.  The tolerance is that of tests/test_gpu_batch.py::test_prepare_strain_against_oracle, applied to the
    difference between the two paths; since both run the same kernels with the same table the difference is in fact
    required to be exactly zero.  Between the calls nothing is cleared or synchronised by the test: each call has to
    cope with what the one before left behind.  The last part checks the claim itself on the driver's books: with the
    outputs allocated beforehand, free device memory is the same before and after a series of calls."""
    import torch
    dev = torch.device("cuda:0")
    cases = [(16384, 4, True), (1 << 20, 1, False), (16384, 4, True), (1 << 19, 2, True)]
    expected, inputs = [], []
    for i, (N, nb, whiten) in enumerate(cases):
        x, inv_asd = _series(N, nb, 1000 + N + nb)
        x_dev = torch.from_numpy(x).to(dev)
        asd_dev = torch.from_numpy(inv_asd).to(dev) if whiten else None
        plan = rbmf.Plan(N, 1024.0, 30.0, 16, 8, w=1, max_candidates=1024, max_triggers=1024, max_batch=nb)
        ref = plan.prepare_strain(x_dev, asd_dev)
        plan.stream.synchronize()
        expected.append(ref.cpu().numpy())
        plan.close()
        inputs.append((x_dev, asd_dev, torch.empty_like(ref)))
    torch.cuda.synchronize()

    stream = torch.cuda.Stream(device=dev)
    # first call on this device (in a fresh process: the one that looks up the array's address), then the rest, all
    # enqueued without waiting in between
    for x_dev, asd_dev, out in inputs:
        got = rbmf.prepare_strain_static(x_dev, asd_dev, out=out, stream=stream)
        assert got is out
    stream.synchronize()
    for (N, nb, whiten), ref, (_, _, out) in zip(cases, expected, inputs):
        got = out.cpu().numpy()
        gain = 2.0 if whiten else 1.0
        bar = 3e-6 * np.abs(ref) + 4e-6 * np.sqrt(N) * gain + 2.0 ** -23 * np.abs(ref).max(axis=1, keepdims=True) * gain
        err = np.abs(got - ref)
        assert (err <= bar).all(), (N, nb, float((err / bar).max()))
        assert np.array_equal(got, ref), (N, nb, float(err.max()))

    # over the limit: refused with a status, nothing launched, the outputs of the earlier calls untouched
    x_big = torch.zeros((3, 1 << 19), dtype=torch.float32, device=dev)
    with pytest.raises(rbmf.RbmfError) as info:
        rbmf.prepare_strain_static(x_big, stream=stream)
    assert info.value.status == rbmf.RBMF_ERR_UNSUPPORTED
    del x_big

    # no allocation: the driver's free-memory figure does not move across a second round of calls
    for x_dev, asd_dev, out in inputs:
        out.zero_()
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(dev)
    for x_dev, asd_dev, out in inputs:
        rbmf.prepare_strain_static(x_dev, asd_dev, out=out, stream=stream)
    stream.synchronize()
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after == free_before, (free_before, free_after)
    for ref, (_, _, out) in zip(expected, inputs):
        assert np.array_equal(out.cpu().numpy(), ref)
