"""GPU parity of afs_pgd_run_conv (per-restart convergence detection; reading G24) against the
oracle's orc_pgd_run_conv: stop counts, returned iterates, best records and the Fig. 4-5 outputs (#unsatisfied, energy,
steps), in the fp64 build exactly and in fp32 within the drift the arithmetic allows."""
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
        "xor": W.xor_dup(104, n=200, m=180).with_run(None, 150, 80),
        "mixed": W.mixed_pb(103, n=200, n_or=600, n_xor=40, n_eo=20, n_amo=20, n_card=12, n_nae=25, n_ek=8,
                            nae_len=(2, 9), ek_len=(3, 30)).with_run(None, 77, 120),
        "long": W.long_pb(105, n=700, n_clauses=900, n_card=7, n_ek=4, long_len=(100, 420)).with_run(None, 40, 130),
    }


@pytest.mark.parametrize("name", ["xor", "mixed", "long"])
@pytest.mark.parametrize("tol", [1e-2, 1e-4])
def test_conv_fp64_build_equals_the_oracle(afs, name, tol):
    import torch
    inst = cases()[name]
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    o = ref.pgd_run_conv(inst, inst.X0, inst.steps, LR, tol, mask=inst.mask)
    for every in (32, 3):                                   # retirement period: results must not depend on it
        P.set_option(2, every)
        X = dev(inst.X0, torch.float64)
        g = P.pgd_run_conv(X, inst.steps, LR, tol, mask=mask)
        torch.cuda.synchronize()
        assert np.array_equal(g["conv_step"].cpu().numpy(), o["conv_step"])
        assert np.abs(X.cpu().numpy() - o["X"]).max() <= 1e-9
        for k in ("best_sat", "best_step", "best_assign", "final_sat"):
            assert np.array_equal(g[k].cpu().numpy(), o[k]), k
        assert np.allclose(g["final_F"].cpu().numpy(), o["final_F"], rtol=1e-11, atol=1e-9)
    if tol >= 1e-2:
        assert (o["conv_step"] >= 0).mean() > 0.1           # the case does exercise stopping
    P.close()


@pytest.mark.parametrize("name", ["xor", "mixed", "long"])
def test_conv_fp32_properties_and_tol_zero(afs, name):
    import torch
    inst = cases()[name]
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    # tol = 0 is afs_pgd_run
    X = dev(inst.X0)
    a = P.pgd_run(X, inst.steps, LR, mask=mask)
    X2 = dev(inst.X0)
    b = P.pgd_run_conv(X2, inst.steps, LR, 0.0, mask=mask)
    assert torch.equal(X, X2) and torch.equal(a["best_sat"], b["best_sat"]) and torch.equal(a["best_assign"], b["best_assign"])
    assert torch.all(b["conv_step"] == -1)
    # tol > 0 in fp32: a stopped restart's X is the plain run's iterate at its stop count; final_sat is its recount
    tol = 1e-3
    X3 = dev(inst.X0)
    c = P.pgd_run_conv(X3, inst.steps, LR, tol, mask=mask)
    cs = c["conv_step"].cpu().numpy()
    o = ref.pgd_run_conv(inst, inst.X0, inst.steps, LR, tol, mask=inst.mask)
    assert np.mean(cs == o["conv_step"]) >= 0.8              # fp32 decides |dX| < tol in fp32: a few borderline restarts
    for t in np.unique(cs[cs >= 0])[:6]:
        Y = dev(inst.X0)
        P.pgd_run(Y, int(t), LR, mask=mask)
        sel = np.nonzero(cs == t)[0]
        assert np.array_equal(Y.cpu().numpy()[sel], X3.cpu().numpy()[sel])
    _, rec = ref.round_count(inst, X3.cpu().numpy().astype(np.float64), want_assign=False)
    assert np.array_equal(rec, c["final_sat"].cpu().numpy())
    Fo, _ = ref.eval_grad(inst, X3.cpu().numpy().astype(np.float64), 2, want_grad=False)
    assert np.all(np.abs(c["final_F"].cpu().numpy() - Fo) <= 1e-4 * np.abs(Fo) + 1e-6 * inst.m)
    with pytest.raises(afs.AfsError):
        P.pgd_run_conv(X3, 5, LR, -1.0)
    P.close()


# ------------------------------------------------------------------------------------------------ per-restart masks
@pytest.mark.parametrize("name", ["mixed", "long"])
def test_per_restart_masks_equal_one_run_per_restart(afs, name):
    """afs_pgd_run_masks (P:L140, L146, L188 (ii)): B different partial assignments in one call.  The definition is the
    oracle's plain run applied to every restart on its own with its own mask; fp64 build, 25 steps."""
    import torch
    inst = cases()[name]
    B = 37
    rng = np.random.default_rng(9)
    masks = np.zeros((B, inst.n), np.int8)
    for b in range(B):
        frac = rng.uniform(0.0, 0.9) if b else 1.0                   # restart 0: everything fixed
        fix = rng.choice(inst.n, size=int(frac * inst.n), replace=False)
        masks[b, fix] = 1 - 2 * rng.integers(0, 2, size=fix.size)
    X0 = inst.X0[:B]
    P = afs.Problem.from_instance(inst)
    X = dev(X0, torch.float64)
    g = P.pgd_run_masks(X, 25, LR, dev(masks))
    torch.cuda.synchronize()
    Xg = X.cpu().numpy()
    for b in range(B):
        o = ref.pgd_run(inst, X0[b:b + 1], 25, LR, mask=masks[b])
        assert np.abs(Xg[b] - o["X"][0]).max() <= 1e-9, b
        assert g["best_sat"][b].item() == o["best_sat"][0] and g["best_step"][b].item() == o["best_step"][0]
        assert np.array_equal(g["best_assign"][b].cpu().numpy(), o["best_assign"][0])
    # fp32: fixed coordinates keep their values bit for bit; equal masks in every row reproduce afs_pgd_run
    Xf = dev(X0)
    P.pgd_run_masks(Xf, 25, LR, dev(masks))
    fixed = masks != 0
    assert np.array_equal(Xf.cpu().numpy()[fixed], masks[fixed].astype(np.float32))
    same = np.tile(masks[5], (B, 1))
    Xa, Xb = dev(X0), dev(X0)
    a = P.pgd_run_masks(Xa, 25, LR, dev(same))
    P.set_option(0, 1)
    b_ = P.pgd_run(Xb, 25, LR, mask=dev(masks[5]))
    if name != "long":        # with long constraints the shared mask is folded, the per-restart one is not: ulp-level drift
        assert torch.equal(Xa, Xb) and torch.equal(a["best_sat"], b_["best_sat"])
    else:
        assert (Xa - Xb).abs().max().item() < 1e-4
    P.close()


@pytest.mark.parametrize("name", ["mixed", "long"])
def test_per_restart_masks_follow_their_restarts_through_retirement(afs, name):
    """A compaction moves restarts to other columns; their masks must move with them.  70 steps with retirement every
    step / every 32 steps / never, rows that are fixed points from the start (everything fixed) in the middle of the
    batch so that the columns behind them shift: fp64 build against one oracle run per restart with its own mask, and
    the fp32 entry bit-identical across the three retirement settings."""
    import torch
    inst = cases()[name]
    B, steps = 70, 70
    rng = np.random.default_rng(21)
    masks = np.zeros((B, inst.n), np.int8)
    for b in range(B):
        frac = 1.0 if b in (0, 3, 40, 41) else rng.uniform(0.0, 0.95)
        fix = rng.choice(inst.n, size=int(frac * inst.n), replace=False)
        masks[b, fix] = 1 - 2 * rng.integers(0, 2, size=fix.size)
    X0 = np.random.default_rng(22).uniform(-1, 1, size=(B, inst.n))
    orc = [ref.pgd_run(inst, X0[b:b + 1], steps, LR, mask=masks[b]) for b in range(B)]
    P = afs.Problem.from_instance(inst)
    md = dev(masks)
    f32 = []
    for every in (0, 1, 32):
        P.set_option(2, every)
        X = dev(X0, torch.float64)
        g = P.pgd_run_masks(X, steps, LR, md)
        torch.cuda.synchronize()
        Xg = X.cpu().numpy()
        for b in range(B):
            o = orc[b]
            assert np.abs(Xg[b] - o["X"][0]).max() <= 1e-9, (every, b)
            assert g["best_sat"][b].item() == o["best_sat"][0] and g["best_step"][b].item() == o["best_step"][0], (every, b)
            assert np.array_equal(g["best_assign"][b].cpu().numpy(), o["best_assign"][0]), (every, b)
        Xf = dev(X0.astype(np.float32))
        gf = P.pgd_run_masks(Xf, steps, LR, md)
        f32.append((Xf.clone(), gf["best_sat"].clone(), gf["best_step"].clone(), gf["best_assign"].clone()))
        fixed = masks != 0
        assert np.array_equal(Xf.cpu().numpy()[fixed], masks[fixed].astype(np.float32)), every
    for r in f32[1:]:
        assert all(torch.equal(x, y) for x, y in zip(f32[0], r))
    P.close()
