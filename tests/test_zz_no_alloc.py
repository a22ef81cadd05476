"""afs_round_count_static, the entry point for callers that cannot allocate device memory when they call.

Such callers exist: a solver loop inside a program whose framework has taken all of HBM into its own pool, a thread
that cannot afford the device-wide synchronisation of cudaMalloc / cudaFree, a plug-in whose host forbids allocations
after set-up.  For them the library keeps the working memory of the round-and-count step in a fixed 16 MiB array that is
part of the library image, shared by every call on that GPU and never cleared between calls.

What is checked here: on two calls in a row (different inputs, the second smaller than the first, so stale contents of
the shared array would show) the integer results equal those of the ordinary afs_round_count exactly -- the tolerance
the other tests use for counts and rounded assignments -- and also the oracle's; the library allocates nothing during
the calls; a request beyond the array is refused with status 9 and leaves the outputs alone.

This file is named to be collected last: `pytest -x` stops at the first failure and must not hide the other tests
behind this one.  It passes alone in a fresh process (its first call does the per-device set-up) and after the others.
"""
import numpy as np
import pytest

import workloads as W
from oracle import ref

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def afs():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m 'not gpu' on CPU boxes)")
    from paper_2606_06656_b200 import build
    build.build()
    import paper_2606_06656_b200 as pkg
    return pkg


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _instance():
    # every constraint type, lengths from 2 to 30, ragged last restart tile
    return W.mixed_pb(311, n=200, n_or=600, n_xor=40, n_eo=20, n_amo=20, n_card=12, n_nae=25, n_ek=8,
                      nae_len=(2, 9), ek_len=(3, 30)).with_run(None, 77, 1)


def test_static_scratch_equals_round_count_on_two_calls_in_a_row(afs):
    import torch
    inst = _instance()
    P = afs.Problem.from_instance(inst)
    rng = np.random.default_rng(5)
    X1 = inst.X0.astype(np.float32).copy()
    X1[0, :6] = [0.0, -0.0, 1.0, -1.0, 1e-30, -1e-30]                       # the rounding rule's edge values (G13)
    X2 = rng.uniform(-1, 1, size=(45, inst.n)).astype(np.float32)          # second call: fewer restarts, other values
    X2[rng.random(X2.shape) < 0.3] = 1.0
    expected = []
    for X in (X1, X2):                                                      # existing path first (it may allocate)
        a, s = P.round_count(dev(X))
        expected.append((a.cpu().numpy(), s.cpu().numpy()))
    # outputs are the caller's: allocate them before the calls, so that nothing allocates while they run
    outs = [(torch.full((X.shape[0], inst.n), 7, dtype=torch.int8, device="cuda"),
             torch.full((X.shape[0],), -5, dtype=torch.int32, device="cuda")) for X in (X1, X2)]
    Xd = [dev(X1), dev(X2)]
    torch.cuda.synchronize()
    ws_before = P.info("workspace_bytes")
    # two calls in a row on one stream; the first one on a device also looks the array's address up (set-up, which
    # may make the driver load the library's device code), so free memory is compared across the second
    P.round_count_static(Xd[0], assign=outs[0][0], sat=outs[0][1])
    free_before = torch.cuda.mem_get_info()[0]
    P.round_count_static(Xd[1], assign=outs[1][0], sat=outs[1][1])
    torch.cuda.synchronize()
    assert P.info("workspace_bytes") == ws_before                                           # the handle's workspace did not grow
    assert torch.cuda.mem_get_info()[0] >= free_before                      # and no device memory left the free pool
    for i, X in enumerate((X1, X2)):
        a, s = outs[i][0].cpu().numpy(), outs[i][1].cpu().numpy()
        assert np.array_equal(s, expected[i][1]), i
        assert np.array_equal(a, expected[i][0]), i
        ao, so = ref.round_count(inst, X.astype(np.float64))
        assert np.array_equal(s, so) and np.array_equal(a, ao), i
    # counts only (assign = NULL), a third call over the second's leftovers
    _, s3 = P.round_count_static(Xd[0], assign=False, sat=outs[0][1].fill_(-5))
    assert np.array_equal(s3.cpu().numpy(), expected[0][1])
    P.close()


def test_static_scratch_refuses_what_does_not_fit(afs):
    import torch
    inst = _instance()
    P = afs.Problem.from_instance(inst)
    # 256-aligned(4 Bp) + 4 n Bp <= 16 MiB: with n = 200 the largest batch is Bp = 20864
    limit = 16 << 20
    Bp_max = (limit // (4 * inst.n + 4)) // 32 * 32
    assert ((4 * Bp_max + 255) // 256) * 256 + 4 * inst.n * Bp_max <= limit
    X = torch.zeros((Bp_max + 1, inst.n), dtype=torch.float32, device="cuda")
    sat = torch.full((Bp_max + 1,), -5, dtype=torch.int32, device="cuda")
    with pytest.raises(afs.AfsError) as e:
        P.round_count_static(X, assign=False, sat=sat)
    assert e.value.status == 9 and "AFS_STATIC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert bool((sat == -5).all())                                          # nothing was enqueued
    # the largest batch that fits is served, and equals the ordinary path (x = 0 rounds to False everywhere)
    _, s_fit = P.round_count_static(X[:Bp_max], assign=False, sat=sat[:Bp_max])
    _, s_ref = P.round_count(X[:Bp_max], want_assign=False)
    assert torch.equal(s_fit, s_ref)
    P.close()
