"""GPU parity of the weighted objective (afs_problem_create_w; PAPER.md L134, L188 (i); reading G25) against the
oracle's orc_eval_grad_w / orc_pgd_run_w."""
import numpy as np
import pytest

import workloads as W
from oracle import ref

pytestmark = pytest.mark.gpu
LR = float(np.float32(0.1))


@pytest.fixture(scope="module")
def afs():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m 'not gpu' on CPU boxes)")
    from paper_2606_06656_b200 import build
    build.build()
    import paper_2606_06656_b200 as pkg
    return pkg


def dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def cases():
    return {
        "mixed": W.mixed_pb(103, n=200, n_or=600, n_xor=40, n_eo=20, n_amo=20, n_card=12, n_nae=25, n_ek=8,
                            nae_len=(2, 9), ek_len=(3, 30)).with_run(None, 45, 20),
        "long": W.long_pb(105, n=700, n_clauses=900, n_card=7, n_ek=4, long_len=(100, 420)).with_run(None, 13, 20),
        "cnf": W.planted_kcnf(101, n=300, m=1260).with_run(None, 70, 20),
    }


def weights_for(inst, seed):
    rng = np.random.default_rng(seed)
    w = rng.uniform(0.25, 3.0, inst.m).astype(np.float32)
    w[rng.random(inst.m) < 0.4] = 1.0            # a good share of unit weights stays on the pull path
    w[rng.integers(0, inst.m)] = 0.0
    return w


@pytest.mark.parametrize("name", ["mixed", "long", "cnf"])
def test_weighted_eval_grad_and_pgd_against_the_oracle(afs, name):
    import torch
    inst = cases()[name]
    w = weights_for(inst, 5)
    P = afs.Problem.from_instance(inst, weights=w)
    Fo, Go, _ = ref.eval_grad_w(inst, w.astype(np.float64), inst.X0.astype(np.float64))
    for dtype, ft, gt in ((torch.float32, 1e-4, 1e-4), (torch.float64, 1e-11, 1e-11)):
        F, G = P.eval_grad(dev(inst.X0, dtype))
        F, G = F.cpu().numpy().astype(np.float64), G.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(F - Fo) <= ft * np.abs(Fo) + (1e-6 if dtype == torch.float32 else 1e-12) * inst.m * 3)
        gmax = np.abs(Go).max(axis=1, keepdims=True)
        assert np.all(np.abs(G - Go) <= gt * gmax)
    mask = None if inst.mask is None else dev(inst.mask)
    o = ref.pgd_run_w(inst, w.astype(np.float64), inst.X0, 20, LR, mask=inst.mask)
    for mode in ((1,) if name == "long" else (1, 2)):
        P.set_option(0, mode)
        X = dev(inst.X0, torch.float64)
        g = P.pgd_run(X, 20, LR, mask=mask)
        assert np.abs(X.cpu().numpy() - o["X"]).max() <= 1e-9
        for k in ("best_sat", "best_step", "best_assign"):
            assert np.array_equal(g[k].cpu().numpy(), o[k]), k
    P.close()


def test_unit_weights_change_nothing(afs):
    import torch
    inst = cases()["mixed"]
    Pa = afs.Problem.from_instance(inst)
    Pb = afs.Problem.from_instance(inst, weights=np.ones(inst.m, np.float32))
    Xa, Xb = dev(inst.X0), dev(inst.X0)
    a = Pa.pgd_run(Xa, 20, LR); b = Pb.pgd_run(Xb, 20, LR)
    assert torch.equal(Xa, Xb) and torch.equal(a["best_sat"], b["best_sat"])
    assert Pa.info("n_pull") == Pb.info("n_pull")
    with pytest.raises(afs.AfsError):
        afs.Problem.from_instance(inst, weights=np.full(inst.m, np.nan, np.float32))
    Pa.close(); Pb.close()


@pytest.mark.parametrize("name", ["mixed", "long", "cnf"])
def test_per_constraint_gradient_magnitudes(afs, name):
    """afs_constraint_grad_l1 = the oracle's gm[k] = sum_b sum_j |dFE_k/dy_j|, unweighted also on a weighted handle; at
    X0 and at a point with 60 % of the coordinates clipped to +-1 (boundary literals of the long constraints)."""
    import torch
    inst = cases()[name]
    rng = np.random.default_rng(6)
    Xc = inst.X0.copy()
    face = rng.random(Xc.shape) < 0.6
    Xc[face] = np.where(Xc[face] < 0, -1.0, 1.0).astype(np.float32)
    for weights in (None, weights_for(inst, 7)):
        P = afs.Problem.from_instance(inst, weights=weights)
        for X in (inst.X0, Xc):
            _, _, gmo = ref.eval_grad_w(inst, None, X.astype(np.float64), want_grad=False, want_gm=True)
            g64 = P.constraint_grad_l1(dev(X, torch.float64)).cpu().numpy()
            assert np.all(np.abs(g64 - gmo) <= 1e-10 * np.maximum(gmo, 1.0)), np.abs(g64 - gmo).max()
            g32 = P.constraint_grad_l1(dev(X)).cpu().numpy().astype(np.float64)
            assert np.all(np.abs(g32 - gmo) <= 1e-4 * np.maximum(gmo, 1e-3) + 1e-5), np.abs(g32 - gmo).max()
        P.close()
