"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's: satisfied counts and rounded assignments bit-exact; fp32 objective
within 1e-4 relative (+1e-6 m absolute, reading G17); gradients within 1e-4 max|grad| per restart (G18); fp64 build
trajectories within 1e-3 over 20 steps (expected ~1e-12)."""
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


# ------------------------------------------------------------------------------------------------ cases
def case_cnf(B=70):      # configs[0]/[3] shape, several variable chunks, ragged restart tail
    return W.planted_kcnf(101, n=300, m=1260).with_run(None, B, 20)


def case_random_cnf(B=64):
    return W.random_kcnf(102, n=50, m=213).with_run(None, B, 20)


def case_mixed(B=45):    # configs[1] shape plus NAE and EK so that all seven types appear
    return W.mixed_pb(103, n=200, n_or=600, n_xor=40, n_eo=20, n_amo=20, n_card=12, n_nae=25, n_ek=8,
                      nae_len=(2, 9), ek_len=(3, 30)).with_run(None, B, 20)


def case_xor(B=96):      # configs[2] shape
    return W.xor_dup(104, n=200, m=180).with_run(None, B, 20)


def case_long(B=13):     # configs[4] shape: clauses + long CARD/EK + mask; lengths straddle the 128-cell rows
    return W.long_pb(105, n=700, n_clauses=900, n_card=7, n_ek=4, long_len=(100, 420)).with_run(None, B, 20)


def case_all_lengths(B=33):
    """every type at lengths that exercise every kernel bucket (pull, 8/16/32/64 padded, two-pass, long rows)"""
    rng = np.random.default_rng(7)
    n = 400
    rows, types, ks = [], [], []
    def add(ty, L, k=0):
        v = rng.choice(n, size=L, replace=False)
        s = 1 - 2 * rng.integers(0, 2, size=L)
        rows.append((s * (v + 1)).astype(np.int32)); types.append(ty); ks.append(k)
    for L in (1, 2, 3, 5, 6, 8, 9, 16, 17, 32, 33, 64, 65, 130, 300):
        add(W.AFS_OR, L); add(W.AFS_XOR, L, int(rng.integers(0, 2)))
    for L in (2, 3, 5, 6, 8, 9, 16, 31, 32, 33, 70, 127, 128, 129, 255, 256, 300):
        add(W.AFS_NAE, L); add(W.AFS_EO, L); add(W.AFS_AMO, L)
        for k in sorted({0, 1, L // 3, L // 2, L - 1, L, L + 1}):
            add(W.AFS_CARD, L, k); add(W.AFS_EK, L, k)
    add(W.AFS_EO, 1); add(W.AFS_AMO, 1); add(W.AFS_CARD, 1, 1); add(W.AFS_EK, 1, 0)
    inst = W.generate._pack("all_lengths", n, rows, types, ks, None, 7)
    inst.with_run(rng, B, 10)
    return inst


CASES = {"cnf": case_cnf, "random_cnf": case_random_cnf, "mixed": case_mixed, "xor": case_xor, "long": case_long,
         "all_lengths": case_all_lengths}


def check_eval(afs, inst, X32, f64=False, sample=None):
    import torch
    P = afs.Problem.from_instance(inst)
    X = dev(X32, torch.float64 if f64 else torch.float32)
    F, G = P.eval_grad(X)
    torch.cuda.synchronize()
    F, G = F.cpu().numpy().astype(np.float64), G.cpu().numpy().astype(np.float64)
    idx = np.arange(X32.shape[0]) if sample is None else sample
    Fo, Go = ref.eval_grad(inst, X32[idx].astype(np.float64), 2)
    ftol = (1e-4 if not f64 else 1e-11) * np.abs(Fo) + (1e-6 if not f64 else 1e-12) * inst.m
    assert np.all(np.abs(F[idx] - Fo) <= ftol), ("F", np.abs(F[idx] - Fo).max(), ftol.min())
    gmax = np.abs(Go).max(axis=1, keepdims=True)
    gtol = (1e-4 if not f64 else 1e-11) * np.maximum(gmax, 1e-30)
    err = np.abs(G[idx] - Go)
    assert np.all(err <= gtol), ("G", (err / gtol).max())
    P.close()
    return err.max(), gmax.max()


# ------------------------------------------------------------------------------------------------ eval_grad
@pytest.mark.parametrize("name", list(CASES))
def test_eval_grad_fp32_parity(afs, name):
    inst = CASES[name]()
    check_eval(afs, inst, inst.X0)


@pytest.mark.parametrize("name", list(CASES))
def test_eval_grad_fp64_build_parity(afs, name):
    inst = CASES[name]()
    check_eval(afs, inst, inst.X0, f64=True)


@pytest.mark.parametrize("name", ["mixed", "long", "all_lengths"])
def test_eval_grad_at_clipped_points(afs, name):
    # PGD iterates sit exactly on the faces x = +-1: leave-one-out must not divide by a vanishing factor
    inst = CASES[name]()
    rng = np.random.default_rng(5)
    X = inst.X0.copy()
    face = rng.random(X.shape) < 0.6
    X[face] = np.sign(X[face])
    X[0] = 1.0; X[1] = -1.0; X[2, ::2] = 0.0
    check_eval(afs, inst, X)


def test_eval_grad_at_the_longest_supported_count_constraints(afs):
    """EK / CARD at the longest length the build accepts (1144) and just below it, every literal strictly inside the
    cube (the largest interior list the item kernel can meet) and with 1, 2, 3 literals on the boundary (every padding of
    its two lists); fp64 build against the oracle.  One literal more is refused at create."""
    rng = np.random.default_rng(31)
    n = 1300
    rows, types, ks = [], [], []
    for L in (1141, 1142, 1143, 1144):
        for ty in (W.AFS_EK, W.AFS_CARD):
            v = rng.choice(n, size=L, replace=False)
            sg = 1 - 2 * rng.integers(0, 2, size=L)
            rows.append((sg * (v + 1)).astype(np.int32)); types.append(ty); ks.append(L // 2 + int(rng.integers(-3, 4)))
    inst = W.generate._pack("longest", n, rows, types, ks, None, 31)
    B = 6
    X = rng.uniform(-0.3, 0.3, size=(B, n))
    for b in range(1, 4):                      # restart b: b literals of every constraint on the boundary
        for r in rows:
            X[b, np.abs(r[:b]) - 1] = rng.choice([-1.0, 1.0], size=b)
    X[4] = np.where(rng.random(n) < 0.5, np.sign(X[4]), X[4])     # about half of everything saturated
    X = X.astype(np.float32)                   # the same representable point for both builds and the oracle
    check_eval(afs, inst, X, f64=True)
    check_eval(afs, inst, X)
    too_long = W.generate._pack("too_long", n, [np.arange(1, 1146, dtype=np.int32)], [W.AFS_CARD], [500], None, 0)
    with pytest.raises(afs.AfsError) as e:
        afs.Problem.from_instance(too_long)
    assert e.value.status == 8


def sub_instance(inst, keep):
    rows = [inst.lits[inst.row_ptr[c]:inst.row_ptr[c + 1]] for c in np.nonzero(keep)[0]]
    return W.generate._pack("sub", inst.n, rows, inst.types[keep], inst.k[keep], None, 0)


@pytest.mark.parametrize("name", ["mixed", "long", "all_lengths"])
def test_eval_grad_per_bucket_subproblems(afs, name):
    # G18 / H7: small-magnitude buckets must not hide behind O(1) clause gradients
    inst = CASES[name]()
    L = inst.lengths()
    groups = {
        "long": L > 64,
        "card_ek": (inst.types == W.AFS_CARD) | (inst.types == W.AFS_EK),
        "eo_amo_nae": (inst.types == W.AFS_EO) | (inst.types == W.AFS_AMO) | (inst.types == W.AFS_NAE),
        "xor": inst.types == W.AFS_XOR,
    }
    for gname, keep in groups.items():
        if keep.sum() == 0:
            continue
        sub = sub_instance(inst, keep)
        check_eval(afs, sub, inst.X0[:9])


# ------------------------------------------------------------------------------------------------ rounding + counts
@pytest.mark.parametrize("name", list(CASES))
def test_round_count_bit_exact(afs, name):
    import torch
    inst = CASES[name]()
    X = inst.X0.copy()
    X[0, :6] = [0.0, -0.0, 1.0, -1.0, 1e-30, -1e-30]          # G13
    P = afs.Problem.from_instance(inst)
    assign, sat = P.round_count(dev(X))
    ao, so = ref.round_count(inst, X.astype(np.float64))
    assert np.array_equal(assign.cpu().numpy(), ao) and np.array_equal(sat.cpu().numpy(), so)
    a64, s64 = P.round_count(dev(X, torch.float64))
    assert np.array_equal(a64.cpu().numpy(), ao) and np.array_equal(s64.cpu().numpy(), so)
    # at Boolean corners too (every literal exactly +-1)
    Xc = np.sign(inst.X0).astype(np.float32)
    _, sat_c = P.round_count(dev(Xc), want_assign=False)
    assert np.array_equal(sat_c.cpu().numpy(), ref.round_count(inst, Xc.astype(np.float64))[1])
    P.close()


# ------------------------------------------------------------------------------------------------ PGD
@pytest.mark.parametrize("name", list(CASES))
def test_pgd_fp64_build_trajectory_20_steps(afs, name):
    import torch
    inst = CASES[name]()
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    orc = ref.pgd_run(inst, inst.X0, 20, LR, mask=inst.mask, want_traj=True)
    for steps in (1, 7, 20):
        X = dev(inst.X0, torch.float64)
        out = P.pgd_run(X, steps, LR, mask=mask)
        torch.cuda.synchronize()
        d = np.abs(X.cpu().numpy() - orc["traj"][steps]).max()
        assert d <= 1e-3, (steps, d)
        assert d <= 1e-9, (steps, d)               # what the arithmetic actually delivers
        # with matching trajectories the integer outputs must match the oracle's run exactly
        o = ref.pgd_run(inst, inst.X0, steps, LR, mask=inst.mask)
        assert np.array_equal(out["best_sat"].cpu().numpy(), o["best_sat"])
        assert np.array_equal(out["best_step"].cpu().numpy(), o["best_step"])
        assert np.array_equal(out["best_assign"].cpu().numpy(), o["best_assign"])
    P.close()


@pytest.mark.parametrize("name", list(CASES))
def test_pgd_fp32_one_step_and_invariants(afs, name):
    import torch
    inst = CASES[name]()
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    # one step against the oracle's step: |dX| <= lr * 1e-4 max|grad| + rounding of x
    X = dev(inst.X0)
    P.pgd_run(X, 1, LR, mask=mask)
    orc1 = ref.pgd_run(inst, inst.X0, 1, LR, mask=inst.mask, want_traj=True)
    X0m = orc1["traj"][0]
    _, Go = ref.eval_grad(inst, X0m, 2)
    tol = LR * 1e-4 * np.abs(Go).max(axis=1, keepdims=True) + 2.5e-7
    assert np.all(np.abs(X.cpu().numpy() - orc1["traj"][1]) <= tol)
    # a 20-step run: properties that hold whatever the fp32 drift (G15)
    X = dev(inst.X0)
    out = P.pgd_run(X, 20, LR, mask=mask)
    torch.cuda.synchronize()
    Xf = X.cpu().numpy()
    assert np.all(np.abs(Xf) <= 1.0)
    if inst.mask is not None:
        fixed = inst.mask != 0
        assert np.array_equal(Xf[:, fixed], np.tile(inst.mask[fixed].astype(np.float32), (inst.B, 1)))
    ba, bs, bt = (out[k].cpu().numpy() for k in ("best_assign", "best_sat", "best_step"))
    assert set(np.unique(ba)) <= {-1, 1}
    _, recount = ref.round_count(inst, ba.astype(np.float64))
    assert np.array_equal(recount, bs)                                   # (i) oracle recount
    _, sat0 = ref.round_count(inst, X0m)
    assert np.all(bs >= sat0) and np.all((bt >= 0) & (bt <= 20))         # (ii)
    # fp32 trajectory stays close to the oracle's over 20 steps on these small cases
    orc = ref.pgd_run(inst, inst.X0, 20, LR, mask=inst.mask)
    assert np.abs(Xf - orc["X"]).max() < 5e-3
    P.close()


@pytest.mark.parametrize("name", ["cnf", "mixed", "long"])
def test_pgd_run_to_run_bit_reproducible_and_resumable(afs, name):
    import torch
    inst = CASES[name]()
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    runs = []
    for _ in range(2):
        X = dev(inst.X0)
        out = P.pgd_run(X, 12, LR, mask=mask)
        torch.cuda.synchronize()
        runs.append((X.cpu().numpy().copy(), {k: v.cpu().numpy().copy() for k, v in out.items() if k != "X"}))
    assert np.array_equal(runs[0][0], runs[1][0])
    for k in runs[0][1]:
        assert np.array_equal(runs[0][1][k], runs[1][1][k])
    # 12 steps == 5 steps then 7 steps on the returned X (G14/G15: X is caller-owned, a second call is resume)
    X = dev(inst.X0)
    a = P.pgd_run(X, 5, LR, mask=mask)
    a_sat = a["best_sat"].cpu().numpy().copy()
    b = P.pgd_run(X, 7, LR, mask=mask)
    assert np.array_equal(X.cpu().numpy(), runs[0][0])
    assert np.array_equal(np.maximum(a_sat, b["best_sat"].cpu().numpy()), runs[0][1]["best_sat"])
    P.close()


def test_pgd_per_iterate_counts_match_history(afs):
    # best_sat / best_step equal max / first argmax of the per-iterate counts, obtained by single-step calls
    import torch
    inst = case_mixed(40)
    P = afs.Problem.from_instance(inst)
    X = dev(inst.X0)
    hist = []
    for t in range(9):
        _, sat = P.round_count(X, want_assign=False)
        hist.append(sat.cpu().numpy().copy())
        P.pgd_run(X, 1, LR)
    _, sat = P.round_count(X, want_assign=False)
    hist.append(sat.cpu().numpy().copy())
    hist = np.stack(hist)
    X2 = dev(inst.X0)
    out = P.pgd_run(X2, 9, LR)
    assert np.array_equal(X2.cpu().numpy(), X.cpu().numpy())
    assert np.array_equal(out["best_sat"].cpu().numpy(), hist.max(axis=0))
    assert np.array_equal(out["best_step"].cpu().numpy(), hist.argmax(axis=0))
    P.close()


def case_no_long(B=37):
    """every type at every length class the tile-resident kernel takes (no CTA-cooperative LONG constraint)"""
    rng = np.random.default_rng(8)
    n = 300
    rows, types, ks = [], [], []
    def add(ty, L, k=0):
        v = rng.choice(n, size=L, replace=False)
        s = 1 - 2 * rng.integers(0, 2, size=L)
        rows.append((s * (v + 1)).astype(np.int32)); types.append(ty); ks.append(k)
    for rep in range(3):
        for L in (1, 2, 3, 4, 5, 6, 8, 9, 16, 17, 32, 33, 64, 65, 130):
            add(W.AFS_OR, L); add(W.AFS_XOR, L, int(rng.integers(0, 2)))
        for L in (2, 3, 5, 6, 8, 9, 16, 31, 32):
            add(W.AFS_NAE, L); add(W.AFS_EO, L); add(W.AFS_AMO, L)
        for L in (1, 2, 7, 16, 17, 32, 33, 48, 49, 64):
            for k in sorted({0, 1, L // 3, L // 2, L - 1, L, L + 1}):
                add(W.AFS_CARD, L, k); add(W.AFS_EK, L, k)
    inst = W.generate._pack("no_long", n, rows, types, ks, None, 8)
    inst.with_run(rng, B, 10)
    return inst


@pytest.mark.parametrize("name,B", [("cnf", 70), ("random_cnf", 64), ("mixed", 45), ("xor", 96), ("no_long", 37),
                                    ("mixed", 300), ("cnf", 1200), ("mixed", 1024), ("xor", 4800)])
def test_resident_kernel_equals_streaming_path(afs, name, B):
    """The one-launch tile-resident kernel runs the same constraint bodies as the per-phase streaming kernels, for
    every cluster size the batch selects, with and without a mask.  fp64 build: iterates within 1e-12 and every integer
    output (best_sat, best_step, best_assign) identical.  fp32: the two kernels inline the bodies into different
    surroundings, so a product may be contracted into an FMA in one and not in the other -- iterates within 2e-6, and
    the integer outputs identical for every restart whose iterates agree to the bit (the large majority)."""
    import torch
    inst = case_no_long(B) if name == "no_long" else CASES[name](B)
    P = afs.Problem.from_instance(inst)
    rng = np.random.default_rng(5)
    mask = np.zeros(inst.n, np.int8)
    fix = rng.choice(inst.n, size=inst.n // 3, replace=False)
    mask[fix] = 1 - 2 * rng.integers(0, 2, size=fix.size)
    for dtype in (torch.float64, torch.float32):
        for steps, mk in ((0, None), (1, None), (12, None), (12, dev(mask))):
            res = {}
            for mode in (1, 2):
                P.set_option(0, mode)
                X = dev(inst.X0, dtype)
                out = P.pgd_run(X, steps, LR, mask=mk)
                torch.cuda.synchronize()
                assert P.info("resident") == (1 if mode == 2 else 0)
                res[mode] = [X.cpu().numpy()] + [out[k].cpu().numpy() for k in ("best_sat", "best_step", "best_assign")]
            dX = np.abs(res[1][0] - res[2][0])
            if dtype == torch.float64:
                assert dX.max() <= 1e-12, dX.max()
                for a, b in zip(res[1][1:], res[2][1:]):
                    assert np.array_equal(a, b)
            else:
                assert dX.max() <= 2e-6, dX.max()
                same = dX.max(axis=1) == 0
                assert same.mean() >= 0.9     # measured on B200: 1.0 in every case of this test
                for a, b in zip(res[1][1:], res[2][1:]):
                    assert np.array_equal(a[same], b[same])
    P.set_option(0, 0)
    X = dev(inst.X0)
    P.pgd_run(X, 3, LR)
    assert P.info("resident") == 1          # auto picks the resident kernel when the instance fits
    P.close()


def test_resident_kernel_refused_when_it_does_not_fit(afs):
    inst = case_long(8)
    P = afs.Problem.from_instance(inst)
    P.set_option(0, 2)
    with pytest.raises(afs.AfsError):
        P.pgd_run(dev(inst.X0), 2, LR)
    P.set_option(0, 0)
    P.pgd_run(dev(inst.X0), 2, LR, mask=dev(inst.mask))
    assert P.info("resident") == 0
    P.close()


def test_profile_read_times_every_kernel_class_of_a_run(afs):
    inst = case_long(8)
    P = afs.Problem.from_instance(inst)
    P.set_option(1, 2)
    X = dev(inst.X0)
    ref_out = P.pgd_run(X, 6, LR, mask=dev(inst.mask))
    prof = P.profile_read()
    assert prof["var"][1] == 3 and prof["var"][0] > 0          # iterations 0, 2, 4
    assert any(k.startswith("long") for k in prof) and "resident" not in prof
    fl = P.profile_flops()                                     # counted by the long kernels of the timed launches
    assert fl and all(k.startswith("long") and v > 0 for k, v in fl.items())
    # never more than the state-independent 6 L K of the constraints, summed over restarts and timed launches
    lens = inst.lengths()[inst.lengths() > 64].astype(float)
    assert sum(fl.values()) <= 6 * (lens * (lens / 2 + 2)).sum() * inst.B * 3
    assert P.profile_flops() == {}
    assert P.profile_read() == {}                              # spans are consumed
    P.set_option(1, 0)
    X2 = dev(inst.X0)
    out = P.pgd_run(X2, 6, LR, mask=dev(inst.mask))
    assert P.profile_read() == {}
    assert np.array_equal(X.cpu().numpy(), X2.cpu().numpy())    # timing does not change results
    assert np.array_equal(ref_out["best_sat"].cpu().numpy(), out["best_sat"].cpu().numpy())
    P.close()
    inst = case_cnf(40)
    P = afs.Problem.from_instance(inst)
    P.set_option(1, 1)
    P.pgd_run(dev(inst.X0), 5, LR)
    prof = P.profile_read()
    assert list(prof) == ["resident"] and prof["resident"][1] == 1
    P.close()


def test_fixed_variables_folded_on_device_equal_a_hand_folded_instance(afs):
    """k_long_fold (literals of the run's fixed variables leave the long constraints, k drops by the fixed true ones)
    against the same folding done by hand on the host: identical fp64 trajectories and counts."""
    import torch
    rng = np.random.default_rng(11)
    n = 500
    rows, types, ks = [], [], []
    for L in (70, 96, 128, 129, 200, 257, 300, 420):
        for ty in (W.AFS_CARD, W.AFS_EK):
            v = rng.choice(n, size=L, replace=False)
            sg = 1 - 2 * rng.integers(0, 2, size=L)
            rows.append((sg * (v + 1)).astype(np.int32)); types.append(ty); ks.append(int(rng.integers(L // 4, 3 * L // 4)))
    mask = np.zeros(n, np.int8)
    fix = rng.choice(n, size=n // 2, replace=False)
    mask[fix] = 1 - 2 * rng.integers(0, 2, size=fix.size)
    frows, fks = [], []
    for lits, ty, k in zip(rows, types, ks):
        mv = mask[np.abs(lits) - 1].astype(int)
        ftrue = int(np.sum((mv != 0) & ((mv < 0) != (lits < 0))))
        keep = lits[mv == 0]
        k2 = k - ftrue
        if ty == W.AFS_CARD:
            k2 = min(max(k2, 0), len(keep) + 1)
        elif k2 < 0 or k2 > len(keep):
            k2 = len(keep) + 1                                   # EK that cannot hold any more
        frows.append(keep); fks.append(k2)
    a = W.generate._pack("fold_a", n, rows, types, ks, None, 11)
    b = W.generate._pack("fold_b", n, frows, types, fks, None, 11)
    X0 = rng.uniform(-1, 1, (21, n))
    Pa, Pb = afs.Problem.from_instance(a), afs.Problem.from_instance(b)
    Xa, Xb = dev(X0), dev(X0)
    oa = Pa.pgd_run(Xa, 15, 0.1, mask=dev(mask))
    ob = Pb.pgd_run(Xb, 15, 0.1, mask=dev(mask))
    assert (Xa - Xb).abs().max().item() < 1e-10
    assert torch.equal(oa["best_sat"], ob["best_sat"]) and torch.equal(oa["best_step"], ob["best_step"])
    assert torch.equal(oa["best_assign"], ob["best_assign"])
    Pa.close(); Pb.close()


def test_host_entry_point_equals_device_entry_point(afs):
    import torch
    inst = case_long(10)
    P = afs.Problem.from_instance(inst)
    Xd = dev(inst.X0)
    d = P.pgd_run(Xd, 6, LR, mask=dev(inst.mask))
    Xh = torch.from_numpy(inst.X0.copy()).pin_memory()
    h = P.pgd_run_host(Xh, 6, LR, mask=inst.mask)
    assert np.array_equal(Xh.numpy(), Xd.cpu().numpy())
    for k in ("best_assign", "best_sat", "best_step"):
        assert np.array_equal(h[k].numpy(), d[k].cpu().numpy())
    assert P.info("launches") > 0
    P.close()


# ------------------------------------------------------------------------------------------------ edge cases
def test_edge_cases(afs):
    import torch
    # no constraints at all
    empty = W.Instance("empty", 5, np.zeros(1, np.int64), np.zeros(0, np.int32), np.zeros(0, np.int32),
                       np.zeros(0, np.int32))
    P = afs.Problem.from_instance(empty)
    X = dev(np.random.default_rng(0).uniform(-1, 1, (3, 5)).astype(np.float32))
    X0 = X.clone()
    F, G = P.eval_grad(X)
    assert torch.all(F == 0) and torch.all(G == 0)
    out = P.pgd_run(X, 4, LR)
    assert torch.equal(X, X0) and torch.all(out["best_sat"] == 0) and torch.all(out["best_step"] == 0)
    P.close()
    # one variable, one unit clause, one restart
    one = W.Instance("one", 1, np.array([0, 1], np.int64), np.array([-1], np.int32), np.array([W.AFS_OR], np.int32),
                     np.zeros(1, np.int32))
    P = afs.Problem.from_instance(one)
    X = dev(np.array([[-0.25]], np.float32))
    F, G = P.eval_grad(X)
    assert abs(F.item() - 0.25) < 1e-7 and abs(G.item() + 1.0) < 1e-7          # FE = y = -x
    out = P.pgd_run(X, 20, LR)
    assert X.item() == 1.0 and out["best_sat"].item() == 1 and out["best_assign"].item() == 1
    P.close()
    # steps = 0 is rounding of X_0; an all-fixed mask keeps the plant and satisfies everything
    inst = case_mixed(5)
    P = afs.Problem.from_instance(inst)
    X = dev(inst.X0)
    out = P.pgd_run(X, 0, LR)
    ao, so = ref.round_count(inst, inst.X0.astype(np.float64))
    assert np.array_equal(out["best_assign"].cpu().numpy(), ao) and np.array_equal(out["best_sat"].cpu().numpy(), so)
    assert np.array_equal(X.cpu().numpy(), inst.X0)
    out = P.pgd_run(X, 3, LR, mask=dev(inst.plant))
    assert torch.all(out["best_sat"] == inst.m) and torch.all(out["best_step"] == 0)
    assert np.array_equal(X.cpu().numpy(), np.tile(inst.plant.astype(np.float32), (5, 1)))
    # argument errors come back as status codes
    with pytest.raises(afs.AfsError):
        P.pgd_run(X, -1, LR)
    with pytest.raises(afs.AfsError):
        P.pgd_run(X, 1, float("nan"))
    P.close()


def test_duplicate_constraints_equal_doubled_step_fp64_build(afs):
    # P:L110 / T11 through the CUDA path
    import torch
    base = W.xor_dup(9, n=64, m=50)
    half = W.Instance("half", base.n, base.row_ptr[:51].copy(), base.lits[:150].copy(), base.types[:50].copy(),
                      base.k[:50].copy())
    X0 = np.random.default_rng(2).uniform(-1, 1, (33, 64))
    Pa, Pb = afs.Problem.from_instance(base), afs.Problem.from_instance(half)
    Xa, Xb = dev(X0), dev(X0)
    Pa.pgd_run(Xa, 25, 0.05)
    Pb.pgd_run(Xb, 25, 0.10)
    assert (Xa - Xb).abs().max().item() < 1e-11
    Pa.close(); Pb.close()


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_full_size_instances_fp64_trajectory_20_steps_on_sampled_restarts(afs, cfg):
    """BASELINE.json: "first-20-step PGD trajectories within 1e-3 in an fp64 verification build", on the full-size
    instances; the oracle runs the sampled restarts one by one (8 restarts x 20 steps; the sample is the first 8)."""
    import torch
    inst = W.config(cfg)
    nb = 8
    X0 = inst.X0[:nb].astype(np.float64)
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    X = dev(X0, torch.float64)
    out = P.pgd_run(X, 20, LR, mask=mask)
    torch.cuda.synchronize()
    o = ref.pgd_run(inst, X0, 20, LR, mask=inst.mask)
    d = np.abs(X.cpu().numpy() - o["X"]).max()
    assert d <= 1e-3, d
    assert d <= 1e-8, d                              # what the arithmetic actually delivers
    assert np.array_equal(out["best_sat"].cpu().numpy(), o["best_sat"])
    assert np.array_equal(out["best_step"].cpu().numpy(), o["best_step"])
    P.close()


# ------------------------------------------------------------------------------------------------ full BASELINE.json sizes
FULL = {0: dict(sample=64, steps=200), 1: dict(sample=48, steps=500), 2: dict(sample=48, steps=1000),
        3: dict(sample=24, steps=300), 4: dict(sample=4, steps=500)}


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_full_size_configs_sampled_parity_and_properties(afs, cfg):
    """At BASELINE.json's sizes, in the launch configuration bench.py times: objective / gradient parity on sampled
    restarts (the oracle computes them one by one), counts bit-exact on all restarts, and the properties of
    afs_pgd_run's outputs that hold at any size."""
    import torch
    inst = W.config(cfg)
    spec = FULL[cfg]
    P = afs.Problem.from_instance(inst)
    rng = np.random.default_rng(cfg)
    sample = np.sort(rng.choice(inst.B, size=min(spec["sample"], inst.B), replace=False))
    check_eval(afs, inst, inst.X0, sample=sample)
    _, sat0 = P.round_count(dev(inst.X0), want_assign=False)
    so = ref.round_count(inst, inst.X0.astype(np.float64), want_assign=False)[1]
    assert np.array_equal(sat0.cpu().numpy(), so)
    mask = None if inst.mask is None else dev(inst.mask)
    X = dev(inst.X0)
    out = P.pgd_run(X, spec["steps"], LR, mask=mask)
    torch.cuda.synchronize()
    Xf = X.cpu().numpy()
    assert np.all(np.abs(Xf) <= 1.0) and np.all(np.isfinite(Xf))
    if inst.mask is not None:
        fixed = inst.mask != 0
        assert np.all(Xf[:, fixed] == inst.mask[fixed].astype(np.float32))
    ba, bs, bt = (out[k].cpu().numpy() for k in ("best_assign", "best_sat", "best_step"))
    _, recount = ref.round_count(inst, ba.astype(np.float64), want_assign=False)
    assert np.array_equal(recount, bs)
    X0m = inst.X0.astype(np.float64)
    if inst.mask is not None:
        X0m[:, fixed] = inst.mask[fixed]
    sat_start = ref.round_count(inst, X0m, want_assign=False)[1]
    assert np.all(bs >= sat_start) and np.all((bt >= 0) & (bt <= spec["steps"]))
    # the returned X is itself an iterate: its count cannot beat the best
    _, sat_end = P.round_count(X, want_assign=False)
    assert np.all(sat_end.cpu().numpy() <= bs)
    # descent happened: mean objective decreased
    Fs, _ = P.eval_grad(dev(X0m.astype(np.float32)), want_G=False)
    Fe, _ = P.eval_grad(X, want_G=False)
    assert Fe.mean().item() < Fs.mean().item()
    P.close()


# ------------------------------------------------------------------------------------------------ retirement of fixed points
@pytest.mark.parametrize("name,B,steps", [("xor", 200, 90), ("xor", 96, 37), ("cnf", 70, 120), ("mixed", 77, 150),
                                          ("long", 45, 130), ("random_cnf", 64, 100)])
def test_retiring_restarts_at_a_fixed_point_changes_no_result(afs, name, B, steps):
    """P:L152-L164 ("idling converged elements waste compute"): the streaming path retires restarts whose iterate did
    not change in a step -- a fixed point of the deterministic PGD map -- and compacts the rest.  Every output must be
    bit-identical to the run that never retires, in fp32 and in the fp64 build, whatever the retirement period."""
    import torch
    inst = CASES[name](B)
    P = afs.Problem.from_instance(inst)
    P.set_option(0, 1)                                   # streaming path
    mask = None if inst.mask is None else dev(inst.mask)
    for dtype in (torch.float32, torch.float64):
        ref_out = None
        for every in (0, 16, 5, 1):
            P.set_option(2, every)
            X = dev(inst.X0, dtype)
            out = P.pgd_run(X, steps, LR, mask=mask)
            torch.cuda.synchronize()
            got = [X.cpu().numpy()] + [out[k].cpu().numpy() for k in ("best_sat", "best_step", "best_assign")]
            if ref_out is None:
                ref_out = got
                moved = True
            else:
                for a, b in zip(ref_out, got):
                    assert np.array_equal(a, b), (str(dtype), every)
        # the case must actually exercise retirement: some restart is at a fixed point by the end
        X = dev(ref_out[0], dtype)
        X1 = X.clone()
        P.set_option(2, 0)
        P.pgd_run(X1, 1, LR, mask=mask)
        frozen = (X1 == X).all(dim=1).float().mean().item()
        if name == "xor":
            assert frozen > 0.2, frozen
    P.set_option(2, 16)
    P.close()


def test_retirement_with_everything_frozen_and_resume(afs):
    """all variables fixed: every restart is at a fixed point after the first step; a second call resumes normally"""
    import torch
    inst = case_mixed(70)
    P = afs.Problem.from_instance(inst)
    P.set_option(0, 1)
    P.set_option(2, 2)
    X = dev(inst.X0)
    out = P.pgd_run(X, 9, LR, mask=dev(inst.plant))
    assert torch.all(out["best_sat"] == inst.m) and torch.all(out["best_step"] == 0)
    assert np.array_equal(X.cpu().numpy(), np.tile(inst.plant.astype(np.float32), (70, 1)))
    X = dev(inst.X0)
    a = P.pgd_run(X, 40, LR)
    Xa = X.clone()
    P.set_option(2, 0)
    X2 = dev(inst.X0)
    b = P.pgd_run(X2, 40, LR)
    assert torch.equal(Xa, X2) and torch.equal(a["best_sat"], b["best_sat"]) and torch.equal(a["best_assign"], b["best_assign"])
    P.close()


@pytest.mark.parametrize("name,B", [("mixed", 77), ("long", 45), ("no_long", 70)])
def test_a_restart_does_not_depend_on_the_restarts_beside_it(afs, name, B):
    """P:L164 / L182: restarts are independent.  Whatever a kernel decides for the 32 restarts of a warp together (which
    body to run, how far a loop goes) must not enter any single restart's arithmetic: a permuted batch, and a batch cut
    to a ragged size, return the same bits restart by restart, on both paths and with 50 steps of drift behind them."""
    import torch
    inst = case_no_long(B) if name == "no_long" else CASES[name](B)
    P = afs.Problem.from_instance(inst)
    mask = None if inst.mask is None else dev(inst.mask)
    perm = np.random.default_rng(3).permutation(B)
    sub = perm[: B - 19]
    for mode in ((1,) if name == "long" else (1, 2)):
        P.set_option(0, mode)
        X = dev(inst.X0)
        o = P.pgd_run(X, 50, LR, mask=mask)
        Xp = dev(inst.X0[perm])
        op = P.pgd_run(Xp, 50, LR, mask=mask)
        Xs = dev(inst.X0[sub])
        os_ = P.pgd_run(Xs, 50, LR, mask=mask)
        torch.cuda.synchronize()
        assert np.array_equal(X.cpu().numpy()[perm], Xp.cpu().numpy())
        assert np.array_equal(X.cpu().numpy()[sub], Xs.cpu().numpy())
        for k in ("best_sat", "best_step", "best_assign"):
            assert np.array_equal(o[k].cpu().numpy()[perm], op[k].cpu().numpy())
            assert np.array_equal(o[k].cpu().numpy()[sub], os_[k].cpu().numpy())
    P.close()
