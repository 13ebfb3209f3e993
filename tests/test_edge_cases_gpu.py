"""Degenerate and boundary cases of the method, each driven through the whole chain (C ABI) and held against the fp64
oracle: a single trace (n = 1), windows that pass nothing (h = 0: every iterate exactly zero) or everything
(h = nt/2), the all-pass band (fmin = 0, fmax = Nyquist: DC and Nyquist bins in B), nine focal points on the automatic
regime (the smallest batch that leaves the streaming GEMV), and the library's state rules (a run keeps its regime while
mk_synthesis runs another one; mk_load_R / eps end a run; overlapping outputs are refused)."""
import numpy as np
import pytest

import oracle
from _util import calibrated, gpu_chain, problem, rel_l2
from paper_2106_04649_b200 import configs

pytestmark = pytest.mark.gpu

TOL_ITER, TOL_FINAL = 2e-5, 1e-4
FINALS = ("f1plus", "f1min", "G", "Gplus", "Gminus")


def _random_problem(n, nt, nfoc, dt, seed, td_samples, fmin, fmax, dx=10.0, eps=2, niter=5):
    """Random non-symmetric causal R, random G_d, traveltimes of `td_samples` (scalar or (lo, hi)) samples; R is scaled by a
    power of two so that the oracle's ||N_1|| / ||N_0|| is about 0.5 (a convergent series that stays above fp32 noise)."""
    rng = np.random.default_rng(seed)
    R = rng.standard_normal((n, n, nt)).astype(np.float32)
    R[:, :, nt // 2:] = 0.0
    Gd = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    Gd[:, :, nt // 4:] = 0.0
    if np.isscalar(td_samples):
        td = np.full((nfoc, n), (td_samples + 0.25) * dt, np.float32)
    else:
        td = ((rng.integers(td_samples[0], td_samples[1], size=(nfoc, n)) + 0.25) * dt).astype(np.float32)
    o = oracle.marchenko(R, Gd, td, dt, dx, fmin, fmax, 2, eps, want=())
    n0, n1 = np.linalg.norm(o["N_iters"][0]), np.linalg.norm(o["N_iters"][1])
    if n0 > 0 and n1 > 0:
        R *= np.float32(2.0 ** np.round(np.log2(0.5 * n0 / n1)))
    else:   # the window passes nothing: scale by the bare synthesis instead
        s = np.linalg.norm(oracle.synthesis(R, oracle.init_field(Gd), dt, oracle.weights(n, dx), *oracle.band(nt, dt, fmin, fmax)[:2]))
        R *= np.float32(2.0 ** np.round(np.log2(0.5 * np.linalg.norm(Gd) / max(s, 1e-300))))
    return R, Gd, td


def _run_both(n, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter, regime=0):
    import torch
    from paper_2106_04649_b200 import binding as B
    ref = oracle.marchenko(R, Gd, td, dt, dx, fmin, fmax, niter, eps)
    nfoc = Gd.shape[0]
    dev = torch.device("cuda:0")
    got = {}
    with B.Marchenko(n, n, nt, dt, dx, fmin, fmax) as mk:
        mk.set_option(B.MK_OPT_EPS_SAMPLES, eps)
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.load_R(torch.from_numpy(R).to(dev))
        mk.begin(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev))
        buf = torch.empty((nfoc, n, nt), dtype=torch.float32, device=dev)
        its = []
        for _ in range(niter):
            mk.step(buf)
            its.append(buf.cpu().numpy().copy())
        got["N_iters"] = np.stack(its) if its else np.zeros((0, nfoc, n, nt), np.float32)
        outs = {nm: torch.empty((nfoc, n, nt), dtype=torch.float32, device=dev) for nm in FINALS}
        mk.finish(outs)
        torch.cuda.synchronize()
        got.update({nm: t.cpu().numpy() for nm, t in outs.items()})
        got["regime"] = int(mk.get_info(B.MK_INFO_REGIME_USED))
    return got, ref


def _assert_parity(got, ref, niter, label, scale_of=None):
    """scale_of: {field: other field} — measure that field's error against the norm of the other one (for a field that
    is a difference of two large terms cancelling to almost nothing, the relative error to itself says nothing)."""
    errs = [rel_l2(got["N_iters"][i], ref["N_iters"][i]) for i in range(niter)]
    fin = {nm: rel_l2(got[nm], ref[nm]) for nm in FINALS}
    for nm, other in (scale_of or {}).items():
        fin[nm] = float(np.linalg.norm(got[nm] - ref[nm]) / np.linalg.norm(ref[other]))
    print(f"\n[{label} regime={got['regime']}] per-iteration max {max(errs) if errs else 0:.2e} " + " ".join(f"{k}={v:.1e}" for k, v in fin.items()))
    assert not errs or max(errs) <= TOL_ITER, errs
    assert max(fin.values()) <= TOL_FINAL, fin


@pytest.mark.parametrize("nt", [64, 2048])
def test_single_trace(nt):
    """n = nshot = nrec = 1: the space integral is one term with weight dx (w[0] = dx when n = 1)."""
    dt, dx, eps, niter = 0.004, 10.0, 2, 5
    fmin, fmax = 10.0, 0.3 / dt
    R, Gd, td = _random_problem(1, nt, 2, dt, 11, nt // 8, fmin, fmax, dx, eps)
    got, ref = _run_both(1, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter)
    _assert_parity(got, ref, niter, f"n=1 nt={nt}")


@pytest.mark.parametrize("nt,nfoc,regime", [(64, 3, 1), (2048, 3, 1), (2048, 12, 3), (4096, 2, 2)])
def test_window_passes_nothing(nt, nfoc, regime):
    """t_d so early that h = clamp(m - eps, 0, nt/2) = 0 for every trace: Theta = 0, every iterate is EXACTLY zero,
    f1plus = T G_d, f1min = 0, and G = p^- + T f2 = R (T G_d) + G_d still needs the first synthesis."""
    n, dt, dx, eps, niter = 9, 0.004, 10.0, 8, 3
    fmin, fmax = 10.0, 0.3 / dt
    R, Gd, td = _random_problem(n, nt, nfoc, dt, 12, 3, fmin, fmax, dx, eps)           # m = 3 < eps = 8
    assert not oracle.window(td, nt, dt, eps).any()
    got, ref = _run_both(n, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter, regime)
    assert not got["N_iters"].any() and not ref["N_iters"].any()
    assert not got["f1min"].any()
    np.testing.assert_array_equal(got["f1plus"], oracle.init_field(Gd).astype(np.float32))
    _assert_parity(got, ref, niter, f"h=0 nt={nt} nfoc={nfoc}")
    assert np.linalg.norm(ref["G"] - Gd) > 1e-3 * np.linalg.norm(Gd)                    # the synthesis term is really there


@pytest.mark.parametrize("nt,nfoc,regime", [(64, 2, 1), (2048, 2, 1), (2048, 10, 3), (4096, 3, 2)])
def test_window_passes_everything(nt, nfoc, regime):
    """t_d beyond the trace: h clamps to nt/2 and Theta passes every sample but j = nt/2 (strict inequality)."""
    n, dt, dx, eps, niter = 7, 0.004, 10.0, 8, 5
    fmin, fmax = 10.0, 0.3 / dt
    R, Gd, td = _random_problem(n, nt, nfoc, dt, 13, nt, fmin, fmax, dx, eps)
    assert (oracle.window(td, nt, dt, eps) == nt // 2).all()
    got, ref = _run_both(n, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter, regime)
    assert not got["N_iters"][:, :, :, nt // 2].any()
    # With an (almost) all-pass window G^- = R f1plus - f1min cancels term by term (-T N_i = R N_{i-1} wherever Theta = 1):
    # what is left is the j = nt/2 sample's trace, 1e-3 of f1min, so its error is measured against f1min
    assert np.linalg.norm(ref["Gminus"]) < 0.05 * np.linalg.norm(ref["f1min"])
    _assert_parity(got, ref, niter, f"h=nt/2 nt={nt} nfoc={nfoc}", scale_of={"Gminus": "f1min"})


@pytest.mark.parametrize("nt,nfoc,regime", [(64, 2, 1), (256, 9, 0), (2048, 2, 1), (2048, 9, 0), (4096, 5, 2)])
def test_all_pass_band_through_the_chain(nt, nfoc, regime):
    """fmin = 0, fmax = Nyquist: B holds every bin, DC and Nyquist included (c_k = 1 there), P_B is the identity."""
    n, dt, dx, eps, niter = 6, 0.004, 10.0, 2, 5
    fmin, fmax = 0.0, 0.5 / dt
    assert oracle.band(nt, dt, fmin, fmax) == (0, nt // 2, nt // 2 + 1)
    R, Gd, td = _random_problem(n, nt, nfoc, dt, 14, (nt // 16, nt // 4), fmin, fmax, dx, eps)
    got, ref = _run_both(n, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter, regime)
    _assert_parity(got, ref, niter, f"all-pass nt={nt} nfoc={nfoc}")


@pytest.mark.parametrize("n,nt", [(40, 256), (130, 2048)])
def test_nine_focal_points_take_the_tensor_regime(n, nt):
    """nfoc = 9 on the automatic regime: the first batch the streaming GEMV does not take."""
    dt, dx, eps, niter = 0.004, 10.0, 4, 6
    fmin, fmax = 10.0, 0.35 / dt
    R, Gd, td = _random_problem(n, nt, 9, dt, 15, (nt // 16, nt // 5), fmin, fmax, dx, eps)
    got, ref = _run_both(n, nt, R, Gd, td, dt, dx, fmin, fmax, eps, niter, regime=0)
    assert got["regime"] == 3
    _assert_parity(got, ref, niter, f"nfoc=9 auto n={n} nt={nt}")


# ---------------------------------------------------------------------------------------------- state rules of the ABI
def _ctx(B, torch, n, nt, dt, dx, fmin, fmax, R, eps):
    mk = B.Marchenko(n, n, nt, dt, dx, fmin, fmax)
    mk.set_option(B.MK_OPT_EPS_SAMPLES, eps)
    mk.load_R(torch.from_numpy(R).cuda())
    return mk


@pytest.mark.parametrize("nfoc_run,nfoc_syn", [(1, 16), (16, 1), (3, 40)])
def test_synthesis_between_steps_does_not_disturb_the_run(nfoc_run, nfoc_syn):
    """include/mk.h: mk_synthesis "does not disturb a run in progress" although it picks its own regime from its own
    nfoc (GEMV for the run and tcgen05 for the synthesis, or the reverse): the interleaved run equals the undisturbed
    one bit for bit, and the synthesis equals one made on a fresh context."""
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt, dt, dx, eps, niter = 40, 256, 0.004, 10.0, 4, 4
    fmin, fmax = 10.0, 0.35 / dt
    R, Gd, td = _random_problem(n, nt, nfoc_run, dt, 21, (16, 50), fmin, fmax, dx, eps)
    rng = np.random.default_rng(3)
    Nin = torch.from_numpy(rng.standard_normal((nfoc_syn, n, nt)).astype(np.float32)).cuda()
    dGd, dtd = torch.from_numpy(Gd).cuda(), torch.from_numpy(td).cuda()
    res = []
    for disturb in (False, True):
        with _ctx(B, torch, n, nt, dt, dx, fmin, fmax, R, eps) as mk:
            S = torch.zeros((nfoc_syn, n, nt), dtype=torch.float32, device="cuda")
            if not disturb:
                mk.synthesis(Nin, S)
            mk.begin(dGd, dtd)
            run_regime = None
            bufs = []
            for i in range(niter):
                if disturb and i in (1, 2):
                    mk.synthesis(Nin, S)
                buf = torch.empty((nfoc_run, n, nt), dtype=torch.float32, device="cuda")
                mk.step(buf)
                r = int(mk.get_info(B.MK_INFO_REGIME_USED))
                run_regime = r if run_regime is None else run_regime
                assert r == run_regime                             # the run kept its regime
                bufs.append(buf)
            if disturb:
                mk.synthesis(Nin, S)
            outs = {nm: torch.empty((nfoc_run, n, nt), dtype=torch.float32, device="cuda") for nm in FINALS}
            mk.finish(outs)
            torch.cuda.synchronize()
            res.append(([b.cpu().numpy() for b in bufs], {k: v.cpu().numpy() for k, v in outs.items()}, S.cpu().numpy()))
    for a, b in zip(res[0][0], res[1][0]):
        np.testing.assert_array_equal(a, b)
    for nm in FINALS:
        np.testing.assert_array_equal(res[0][1][nm], res[1][1][nm])
    np.testing.assert_array_equal(res[0][2], res[1][2])


def test_reload_and_new_eps_end_a_run_and_the_next_run_uses_them():
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt, dt, dx, eps, niter = 12, 128, 0.004, 10.0, 3, 3
    fmin, fmax = 10.0, 0.3 / dt
    R, Gd, td = _random_problem(n, nt, 2, dt, 31, (10, 30), fmin, fmax, dx, eps)
    R2 = R.copy()
    R2[4:7] *= np.float32(0.5)
    dGd, dtd = torch.from_numpy(Gd).cuda(), torch.from_numpy(td).cuda()
    outs = {nm: torch.empty((2, n, nt), dtype=torch.float32, device="cuda") for nm in FINALS}
    with _ctx(B, torch, n, nt, dt, dx, fmin, fmax, R, eps) as mk:
        mk.run(dGd, dtd, niter, outs)
        mk.begin(dGd, dtd)
        mk.step_contract()
        with pytest.raises(B.MkError) as e:                         # refused between the two halves of a step
            mk.load_R(torch.from_numpy(R2[4:7]).cuda(), 4)
        assert e.value.code == B.MK_ERR_STATE
        mk.step_post()
        mk.load_R(torch.from_numpy(R2[4:7]).cuda(), 4)             # replaces shots 4..6; the run in progress is over
        with pytest.raises(B.MkError) as e:
            mk.step()
        assert e.value.code == B.MK_ERR_STATE
        with pytest.raises(B.MkError):
            mk.finish(outs)
        mk.run(dGd, dtd, niter, outs)
        torch.cuda.synchronize()
        a = {k: v.cpu().numpy() for k, v in outs.items()}
        mk.begin(dGd, dtd)
        mk.set_option(B.MK_OPT_EPS_SAMPLES, eps)                   # same value: nothing changes
        mk.step()
        mk.set_option(B.MK_OPT_EPS_SAMPLES, eps + 2)               # new window: ends the run
        with pytest.raises(B.MkError):
            mk.step()
        mk.run(dGd, dtd, niter, outs)
        torch.cuda.synchronize()
        c = {k: v.cpu().numpy() for k, v in outs.items()}
    ref_a = oracle.marchenko(R2, Gd, td, dt, dx, fmin, fmax, niter, eps)
    ref_c = oracle.marchenko(R2, Gd, td, dt, dx, fmin, fmax, niter, eps + 2)
    for nm in FINALS:
        assert rel_l2(a[nm], ref_a[nm]) <= TOL_FINAL, nm
        assert rel_l2(c[nm], ref_c[nm]) <= TOL_FINAL, nm
    assert rel_l2(a["G"], ref_c["G"]) > 1e-3                        # the two windows really differ


def test_overlapping_outputs_are_refused():
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt, dt, dx = 8, 64, 0.004, 10.0
    rng = np.random.default_rng(7)
    R = (0.01 * rng.standard_normal((n, n, nt))).astype(np.float32)
    Gd = torch.from_numpy(rng.standard_normal((2, n, nt)).astype(np.float32)).cuda()
    td = torch.full((2, n), 0.08, dtype=torch.float32, device="cuda")
    f = lambda: torch.empty((2, n, nt), dtype=torch.float32, device="cuda")
    with _ctx(B, torch, n, nt, dt, dx, 10.0, 100.0, R, 2) as mk:
        a, b, c = f(), f(), f()
        for bad in ({"f1plus": a, "f1min": a}, {"f1plus": Gd}, {"f1plus": a, "G": a}, {"f1min": b, "Gminus": b},
                    {"f1plus": a, "f1min": b, "N_last": b}):
            with pytest.raises(B.MkError) as e:
                mk.run(Gd, td, 2, bad)
            assert e.value.code == B.MK_ERR_INVALID_ARG
        mk.run(Gd, td, 2, {"f1plus": a, "f1min": b, "G": c, "Gplus": c, "Gminus": c, "N_last": c})   # sharing among the rest is allowed
        mk.begin(Gd, td)
        mk.step()
        lib_plus = f()
        mk.finish({"f1plus": lib_plus})
        with pytest.raises(B.MkError):
            big = torch.empty((2 * 2 * n * nt,), dtype=torch.float32, device="cuda")
            mk.finish({"f1plus": big[: 2 * n * nt].view(2, n, nt), "f1min": big[n * nt: n * nt + 2 * n * nt].view(2, n, nt)})
        torch.cuda.synchronize()
        ref = oracle.marchenko(R, Gd.cpu().numpy(), td.cpu().numpy(), dt, dx, 10.0, 100.0, 1, 2)
        assert rel_l2(lib_plus.cpu().numpy(), ref["f1plus"]) <= TOL_FINAL


@pytest.mark.parametrize("k,n,nt,nfoc", [(2, 70, 512, 70), (3, 150, 2048, 19), (4, 60, 1024, 33), (1, 300, 256, 5), (1, 129, 512, 1)])
def test_tiled_rhat_layout_equals_the_row_major_one(k, n, nt, nfoc):
    """MK_OPT_RHAT_LAYOUT = 1: R^ stored in 16 KB boxes of [128 receivers][16 shots] for the tcgen05 contraction (one bulk
    copy per box instead of a TMA box of 128 rows 2 MB apart).  Same kernel, same arithmetic, another address map: the
    whole chain must equal the row-major regime-3 run BIT FOR BIT and meet the oracle; receiver counts that are no
    multiple of 128 (padded tile rows), ragged focal batches, one focal point (which takes regime 3 here as well)."""
    import oracle
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal="single:400" if nfoc == 1 else "fan:250", niter=5))
    R, Gd, td = problem(cfg)
    a = gpu_chain(cfg, R, Gd, td, regime=3, rhat_layout=0)
    b = gpu_chain(cfg, R, Gd, td, regime=0, rhat_layout=1)
    assert b["regime_used"] == 3
    for nm in ("N_iters", "f1plus", "f1min", "G", "Gplus", "Gminus"):
        assert np.array_equal(a[nm], b[nm]), nm
    ref = oracle.marchenko(R, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, cfg.niter, cfg.eps)
    errs = [rel_l2(b["N_iters"][i], ref["N_iters"][i]) for i in range(cfg.niter)]
    fin = max(rel_l2(b[nm], ref[nm]) for nm in ("f1plus", "f1min", "G", "Gplus", "Gminus"))
    print(f"\n[tiled R^ n={n} nt={nt} nfoc={nfoc}] bit-identical to the row-major layout; per-iteration max {max(errs):.2e}, finals {fin:.2e}")
    assert np.linalg.norm(ref["N_iters"][-1]) > 0          # the series is alive: the bounds are not vacuous
    assert max(errs) <= 2e-5 and fin <= 1e-4


def test_tiled_rhat_layout_rules():
    import torch
    from paper_2106_04649_b200 import binding as B
    cfg = configs.scaled(1, n=40, nt=64, nfoc=2, focal="fan:250", niter=1)
    R, Gd, td = problem(cfg)
    dev = torch.device("cuda:0")
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax) as mk:
        mk.set_option(B.MK_OPT_RHAT_LAYOUT, 1)
        mk.set_option(B.MK_OPT_REGIME, 1)
        mk.load_R(torch.from_numpy(R).to(dev))
        with pytest.raises(B.MkError):                      # the streaming GEMV cannot read the tiled layout
            mk.begin(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev))
        with pytest.raises(B.MkError):                      # laid out at ingest
            mk.set_option(B.MK_OPT_RHAT_LAYOUT, 0)
        with pytest.raises(B.MkError):
            mk.set_option(B.MK_OPT_RHAT_FORMAT, 1)
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(0, 20)) as mk:
        with pytest.raises(B.MkError):                      # plain contexts only
            mk.set_option(B.MK_OPT_RHAT_LAYOUT, 1)


def test_sync_and_row_ingest_argument_rules():
    """mk_sync_* and mk_load_R_rows refuse what they cannot do (MK_ERR_*), and a one-rank barrier is a no-op."""
    import torch
    from paper_2106_04649_b200 import binding as B
    cfg = configs.scaled(1, n=40, nt=64, nfoc=2, focal="fan:250", niter=1)
    R, Gd, td = problem(cfg)
    dev = torch.device("cuda:0")
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax) as mk:
        with pytest.raises(B.MkError):
            mk.sync_barrier()                                # before mk_sync_create
        with pytest.raises(B.MkError):
            mk.sync_flags()
        with pytest.raises(B.MkError):
            mk.sync_create(2, 2)                             # rank out of range
        with pytest.raises(B.MkError):
            mk.sync_create(0, 9)                             # more ranks than flag slots
        mk.sync_create(0, 1)
        mk.sync_barrier()                                    # one rank: nothing to wait for
        mk.sync_create(0, 2)
        assert mk.sync_flags() != 0
        with pytest.raises(B.MkError):
            mk.sync_barrier()                                # two ranks, peers not attached
        with pytest.raises(B.MkError):
            mk.sync_attach([None, None])                     # the peer's flag array is missing
        # mk_load_R_rows on an unsharded context is mk_load_R
        mk.load_R_rows(torch.from_numpy(R).to(dev))
        a = torch.empty((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev)
        mk.run(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev), 1, {"G": a})
        torch.cuda.synchronize()
    ref = gpu_chain(cfg, R, Gd, td, niter=1, keep_iters=False, outputs=("G",))
    assert np.array_equal(a.cpu().numpy(), ref["G"])
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, streamed=(10, 10)) as mk:
        with pytest.raises(B.MkError):                       # out-of-core R^: rows do not all live on the device
            mk.load_R_rows(torch.from_numpy(R).to(dev))
