"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element on the same seeded
inputs.  Tolerances are BASELINE.json north_star's: relative L2 error <= 2e-5 per iteration and <= 1e-4 on the
final fields.  Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest

import oracle
from paper_2106_04649_b200 import configs, gen
from _util import calibrated, gpu_chain, problem, rel_l2

pytestmark = pytest.mark.gpu

TOL_ITER, TOL_FINAL = 2e-5, 1e-4
FINALS = ("f1plus", "f1min", "G", "Gplus", "Gminus")


def _oracle_chain(cfg, R, Gd, td, niter=None):
    return oracle.marchenko(R, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, cfg.niter if niter is None else niter, cfg.eps)


def _check_chain(cfg, regime, niter=None, focs=None):
    R, Gd, td = problem(cfg, focs)
    ref = _oracle_chain(cfg, R, Gd, td, niter)
    got = gpu_chain(cfg, R, Gd, td, niter=niter, regime=regime)
    errs = [rel_l2(got["N_iters"][i], ref["N_iters"][i]) for i in range(ref["N_iters"].shape[0])]
    ferr = {nm: rel_l2(got[nm], ref[nm]) for nm in FINALS}
    print(f"\n[{cfg.name} n={cfg.n} nt={cfg.nt} nfoc={Gd.shape[0]} regime={got['regime_used']}] per-iter max {max(errs):.2e} "
          + " ".join(f"{k}={v:.1e}" for k, v in ferr.items()))
    assert max(errs) <= TOL_ITER, errs
    for nm, e in ferr.items():
        assert e <= TOL_FINAL, (nm, e)
    return got, ref


# ---------------------------------------------------------------- bare synthesis
@pytest.mark.parametrize("n,nt,nfoc,regime", [(5, 32, 3, 0), (20, 64, 1, 1), (20, 64, 12, 2), (20, 64, 12, 3),
                                               (6, 2048, 3, 0), (6, 4096, 2, 0), (5, 4096, 9, 0)])   # register-resident transforms, all-pass band
def test_delta_spike_shift(n, nt, nfoc, regime):
    import torch
    from paper_2106_04649_b200 import binding as B
    dt, dx, q = 0.5, 2.0, 5
    w = np.full(n, dx)
    w[0] = w[-1] = dx / 2
    R = np.zeros((n, n, nt), np.float32)
    for s in range(n):
        R[s, s, q] = 1.0 / (w[s] * dt)
    rng = np.random.default_rng(1)
    N = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    with B.Marchenko(n, n, nt, dt, dx, 0.0, 1.0 / (2 * dt)) as mk:
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.load_R(torch.from_numpy(R).cuda())
        S = torch.empty((nfoc, n, nt), dtype=torch.float32, device="cuda")
        mk.synthesis(torch.from_numpy(N).cuda(), S)
        S = S.cpu().numpy()
    assert rel_l2(S, np.roll(N, q, axis=-1)) < 2e-6


@pytest.mark.parametrize("n,nt,nfoc,regime", [
    (37, 128, 1, 1), (37, 128, 3, 1), (37, 128, 8, 1),           # GEMV, ragged rows
    (37, 128, 5, 2), (150, 64, 70, 2), (130, 256, 129, 2),        # FFMA GEMM, ragged M / N tiles
    (37, 128, 5, 3), (150, 64, 70, 3), (130, 256, 129, 3), (260, 64, 140, 3),   # tcgen05 3xTF32, ragged M / N / K tiles
    (300, 64, 20, 3), (257, 64, 64, 3),                           # two M tiles per B' tile, odd tile count / one-row last tile
    (16, 16, 2, 0), (33, 4096, 9, 0),                             # smallest / longest traces
    (24, 2048, 11, 0), (24, 2048, 1, 1), (20, 2048, 3, 1), (20, 4096, 1, 1), (18, 4096, 16, 3),   # register-resident transforms
])
def test_synthesis_random_vs_oracle(n, nt, nfoc, regime):
    import torch
    from paper_2106_04649_b200 import binding as B
    dt, dx = 0.004, 10.0
    fmax = 0.4 / dt
    rng = np.random.default_rng(n * 1000 + nfoc)
    R = rng.standard_normal((n, n, nt)).astype(np.float32)     # non-symmetric in (s, r): a transposed operand fails
    N = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    N[:, :, nt // 3:] = 0.0                                      # keeps the direct oracle cheap
    klo, khi, nb = oracle.band(nt, dt, 10.0, fmax)
    ref = oracle.synthesis(R, N.astype(np.float64), dt, oracle.weights(n, dx), klo, khi)
    with B.Marchenko(n, n, nt, dt, dx, 10.0, fmax) as mk:
        assert int(mk.get_info(B.MK_INFO_NB)) == nb and int(mk.get_info(B.MK_INFO_KLO)) == klo
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.load_R(torch.from_numpy(R).cuda())
        S = torch.empty((nfoc, n, nt), dtype=torch.float32, device="cuda")
        mk.synthesis(torch.from_numpy(N).cuda(), S)
        S = S.cpu().numpy()
    e = rel_l2(S, ref)
    print(f"\n[synthesis n={n} nt={nt} nfoc={nfoc} regime={regime}] rel L2 {e:.2e}")
    assert e <= TOL_ITER


# ---------------------------------------------------------------- whole chain, reduced copies of the configs
@pytest.mark.parametrize("k,n,nt,nfoc,regime", [
    (0, 40, 256, 1, 1), (1, 70, 512, 4, 1), (1, 70, 512, 4, 2), (2, 70, 512, 70, 2), (3, 90, 512, 19, 2),
    (4, 60, 1024, 33, 2), (2, 70, 512, 70, 3), (3, 90, 512, 19, 3), (4, 60, 1024, 33, 3),
    # nt = 2048 / 4096: the register-resident transform kernels (mk_fft_fast.cu), ragged focal groups
    (1, 30, 2048, 1, 1), (2, 30, 2048, 30, 2), (3, 26, 2048, 11, 3), (4, 24, 4096, 11, 2), (4, 24, 4096, 5, 1),
])
def test_chain_reduced_configs(k, n, nt, nfoc, regime):
    focal = "single:400" if nfoc == 1 else ("line:300" if nfoc == n else "fan:250")
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal=focal, niter=8))
    _check_chain(cfg, regime)


def test_transform_paths_agree():
    """MK_OPT_FFT_PATH: the generic shared-memory kernels and the register-resident ones are two implementations of
    the same steps; both must meet the oracle (checked above) and therefore agree with each other to rounding."""
    cfg = calibrated(configs.scaled(3, n=26, nt=2048, nfoc=11, focal="fan:250", niter=6))
    R, Gd, td = problem(cfg)
    a = gpu_chain(cfg, R, Gd, td, regime=2, fft_path=1)
    b = gpu_chain(cfg, R, Gd, td, regime=2, fft_path=2)
    for nm in FINALS + ("N_iters",):
        assert rel_l2(a[nm], b[nm]) <= 5e-6, nm


def test_config0_full_chain():
    got, ref = _check_chain(configs.get(0), regime=0)
    assert got["regime_used"] == 1


def test_config0_host_api_and_run_match_steps():
    cfg = configs.get(0)
    R, Gd, td = problem(cfg)
    a = gpu_chain(cfg, R, Gd, td, keep_iters=True)
    b = gpu_chain(cfg, R, Gd, td, keep_iters=False)
    c = gpu_chain(cfg, R, Gd, td, host_api=True)
    for nm in FINALS:
        np.testing.assert_array_equal(a[nm], b[nm])
        np.testing.assert_array_equal(a[nm], c[nm])
    np.testing.assert_array_equal(a["N_iters"][-1], b["N_last"])
    np.testing.assert_array_equal(b["N_last"], c["N_last"])


@pytest.mark.parametrize("niter", [1, 2, 3])
def test_host_api_equals_device_api_for_odd_and_even_step_counts(niter):
    """mk_run_host copies the accumulator that the last step does not touch (f1plus after an odd number of steps, f1min after
    an even one) to the host while that step runs: both parities, and a single step, give the bits of mk_run."""
    cfg = calibrated(configs.scaled(2, n=40, nt=256, nfoc=5, focal="fan:300", niter=niter))
    R, Gd, td = problem(cfg)
    b = gpu_chain(cfg, R, Gd, td, keep_iters=False)
    c = gpu_chain(cfg, R, Gd, td, host_api=True)
    for nm in FINALS + ("N_last",):
        assert np.abs(b[nm]).max() > 0, nm
        np.testing.assert_array_equal(b[nm], c[nm])


def test_image_matches_oracle():
    """NEXT-1: double-focusing image of a small multi-focal run against the oracle's definition."""
    import torch
    from paper_2106_04649_b200 import binding as B
    cfg = calibrated(configs.scaled(2, n=48, nt=256, nfoc=48, focal="line:300", niter=6))
    R, Gd, td = problem(cfg)
    ref = _oracle_chain(cfg, R, Gd, td)
    img_ref = oracle.image(ref["Gminus"], ref["f1plus"], cfg.dt, cfg.dx)
    dev = torch.device("cuda:0")
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax) as mk:
        mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
        mk.load_R(torch.from_numpy(R).to(dev))
        outs = {"Gminus": torch.empty((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev)}
        mk.run(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev), cfg.niter, outs)
        img = torch.empty(cfg.nfoc, dtype=torch.float32, device=dev)
        mk.image(outs["Gminus"], img)
        img = img.cpu().numpy()
    e = rel_l2(img, img_ref)
    print(f"\n[image nfoc={cfg.nfoc}] rel L2 {e:.2e}")
    assert e <= TOL_FINAL


# ---------------------------------------------------------------- receiver-row sharding (section 8(e), NEXT-3)

def _sharded_vs_oracle(ref, world, n, its, outs, niter):
    """Every rank's own receiver rows of every iterate and every final field against the fp64 oracle (the parity bar
    proper; the comparison with the unsharded CUDA run beside it is the bit-level regression check)."""
    from paper_2106_04649_b200 import shard
    worst_it = worst_fin = 0.0
    for g in range(world):
        rows = shard.row_slice(n, g, world)
        sl = slice(rows.start, rows.stop)
        for i in range(niter):
            worst_it = max(worst_it, rel_l2(its[g][i][:, sl], ref["N_iters"][i][:, sl]))
        for nm in FINALS:
            worst_fin = max(worst_fin, rel_l2(outs[g][nm].cpu().numpy()[:, sl], ref[nm][:, sl]))
    return worst_it, worst_fin

@pytest.mark.parametrize("k,n,nt,nfoc,regime,world", [(1, 37, 512, 3, 1, 2), (3, 45, 512, 19, 2, 3), (3, 150, 2048, 19, 3, 3)])
def test_row_sharded_contexts_reproduce_the_single_context(k, n, nt, nfoc, regime, world):
    """`world` row-sharded contexts in one process, stepped in lock-step with the operand rows copied between them
    (shard.exchange_in_process — what the NCCL all-gather does across GPUs): every rank's receiver rows of every iterate
    and every final field must meet the oracle to the north_star tolerance and equal the unsharded run."""
    import torch
    from paper_2106_04649_b200 import binding as B, shard
    focal = "single:400" if nfoc == 1 else "fan:250"
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal=focal, niter=6))
    R, Gd, td = problem(cfg)
    whole = gpu_chain(cfg, R, Gd, td, regime=regime)
    ref = _oracle_chain(cfg, R, Gd, td)
    dev = torch.device("cuda:0")
    dR, dGd, dtd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (R, Gd, td))
    mks = []
    try:
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            mk = B.Marchenko(n, n, nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(rows.start, len(rows)))
            mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
            mk.set_option(B.MK_OPT_REGIME, regime)
            mk.load_R(dR)                                   # same full chunk on every rank; the library keeps its rows
            mks.append(mk)
        # a contraction on rows that were not exchanged must fail loudly
        mks[0].begin(dGd, dtd)
        with pytest.raises(B.MkError):
            mks[0].step()
        with pytest.raises(B.MkError):
            mks[0].run(dGd, dtd, 1, {})
        for mk in mks:
            mk.begin(dGd, dtd)
        shard.exchange_in_process(mks, 0)
        its = [[] for _ in mks]
        bufs = [torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for _ in mks]
        for _ in range(cfg.niter):
            for g, mk in enumerate(mks):
                mk.step(bufs[g])
                its[g].append(bufs[g].cpu().numpy().copy())
            shard.exchange_in_process(mks, 0)
        outs = [{nm: torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for nm in FINALS} for _ in mks]
        for g, mk in enumerate(mks):
            mk.finish({nm: outs[g][nm] for nm in ("f1plus", "f1min", "G")})
        for name, field in (("Gminus", B.MK_FIELD_GMINUS), ("Gplus", B.MK_FIELD_GPLUS)):
            for mk in mks:
                mk.finish_prepare(field)
            shard.exchange_in_process(mks, 1)
            for g, mk in enumerate(mks):
                mk.finish_complete(field, outs[g][name])
        torch.cuda.synchronize()
        worst = 0.0
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            sl = slice(rows.start, rows.stop)
            for i in range(cfg.niter):
                worst = max(worst, rel_l2(its[g][i][:, sl], whole["N_iters"][i][:, sl]))
            for nm in FINALS:
                worst = max(worst, rel_l2(outs[g][nm].cpu().numpy()[:, sl], whole[nm][:, sl]))
        worst_it, worst_fin = _sharded_vs_oracle(ref, world, n, its, outs, cfg.niter)
        print(f"\n[row-sharded {world} x, n={n} nt={nt} nfoc={nfoc} regime={regime}] worst deviation from the single context {worst:.1e}; "
              f"each rank's rows against the oracle: per-iteration {worst_it:.2e}, finals {worst_fin:.2e}")
        assert worst <= 1e-6
        assert worst_it <= TOL_ITER and worst_fin <= TOL_FINAL
    finally:
        for mk in mks:
            mk.close()


# ---------------------------------------------------------------- error behaviour and degenerate runs through the C ABI
def test_error_paths_and_degenerate_runs():
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt, dt, dx = 12, 64, 0.004, 10.0
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(5)
    R = torch.from_numpy(rng.standard_normal((n, n, nt)).astype(np.float32)).to(dev)
    Gd = torch.from_numpy(rng.standard_normal((2, n, nt)).astype(np.float32)).to(dev)
    td = torch.full((2, n), 0.05, dtype=torch.float32, device=dev)
    outs = {nm: torch.empty((2, n, nt), dtype=torch.float32, device=dev) for nm in ("f1plus", "f1min", "G")}
    with B.Marchenko(n, n, nt, dt, dx, 10.0, 100.0) as mk:
        mk.load_R(R[:5].contiguous(), 0)
        with pytest.raises(B.MkError) as e:                      # a run before every shot is loaded is an error, not a silent zero
            mk.run(Gd, td, 2, outs)
        assert e.value.code == B.MK_ERR_STATE
        with pytest.raises(B.MkError):
            mk.load_R(R[:5].contiguous(), 9)                     # shot range past the end
        with pytest.raises(B.MkError):
            mk.step()                                            # step before begin
        mk.load_R(R[5:].contiguous(), 5)
        with pytest.raises(B.MkError):
            mk.set_option(B.MK_OPT_FFT_PATH, 2)                  # register-resident transforms need nt = 2048 / 4096
        mk.set_option(B.MK_OPT_REGIME, 1)
        Gd9 = torch.zeros((9, n, nt), dtype=torch.float32, device=dev)
        with pytest.raises(B.MkError):
            mk.begin(Gd9, torch.zeros((9, n), dtype=torch.float32, device=dev))   # the streaming GEMV takes at most 8 focal points
        mk.set_option(B.MK_OPT_REGIME, 0)
        with pytest.raises(B.MkError):
            mk.run(Gd, td, 0, {"N_last": outs["G"]})             # N_last of a run without iterations
        # niter = 0: f1plus = N_{-1} = T G_d, f1min = 0, G = p^- + T f2 = G_d   [PAPER.md:19, 67, 74-75]
        mk.run(Gd, td, 0, outs)
        torch.cuda.synchronize()
        g = Gd.cpu().numpy()
        np.testing.assert_array_equal(outs["f1plus"].cpu().numpy(), np.roll(g[..., ::-1], 1, axis=-1))
        assert float(outs["f1min"].abs().max()) == 0.0
        assert rel_l2(outs["G"].cpu().numpy(), g) < 1e-6
        # the context stays usable after errors
        mk.run(Gd, td, 1, outs)
        torch.cuda.synchronize()
        assert np.isfinite(outs["G"].cpu().numpy()).all()


@pytest.mark.parametrize("k,n,nt,nfoc,regime,world", [(1, 37, 512, 3, 1, 2), (3, 45, 512, 19, 2, 3), (3, 150, 2048, 19, 3, 3)])
def test_row_sharded_with_fused_peer_stores(k, n, nt, nfoc, regime, world):
    """The exchange fused into the producing kernels (mk_operand_attach): no copies between the contexts, every rank's
    k_fwd / k_post stores its rows into all the others' operands; lock-step order contract -> post, as the barriers of
    shard.run_row_sharded_fused enforce across processes."""
    import torch
    from paper_2106_04649_b200 import binding as B, shard
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal="fan:250", niter=5))
    R, Gd, td = problem(cfg)
    whole = gpu_chain(cfg, R, Gd, td, regime=regime)
    ref = _oracle_chain(cfg, R, Gd, td)
    dev = torch.device("cuda:0")
    dR, dGd, dtd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (R, Gd, td))
    mks = []
    try:
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            mk = B.Marchenko(n, n, nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(rows.start, len(rows)))
            mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
            mk.set_option(B.MK_OPT_REGIME, regime)
            mk.load_R(dR)
            mks.append(mk)
        shard.attach_in_process(mks, nfoc)
        for mk in mks:
            mk.begin(dGd, dtd)
        for mk in mks:
            mk.operand_exchanged(0)
        bufs = [torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for _ in mks]
        its = [[] for _ in mks]
        for _ in range(cfg.niter):
            for mk in mks:
                mk.step_contract()
            for g, mk in enumerate(mks):
                mk.step_post(bufs[g])
                its[g].append(bufs[g].cpu().numpy().copy())
            for mk in mks:
                mk.operand_exchanged(0)
        outs = [{nm: torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for nm in FINALS} for _ in mks]
        for g, mk in enumerate(mks):
            mk.finish({nm: outs[g][nm] for nm in ("f1plus", "f1min", "G")})
        for name, field in (("Gminus", B.MK_FIELD_GMINUS), ("Gplus", B.MK_FIELD_GPLUS)):
            for mk in mks:
                mk.finish_prepare(field)
            for mk in mks:
                mk.operand_exchanged(1)
            for g, mk in enumerate(mks):
                mk.finish_complete(field, outs[g][name])
        torch.cuda.synchronize()
        worst = 0.0
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            sl = slice(rows.start, rows.stop)
            for i in range(cfg.niter):
                worst = max(worst, rel_l2(its[g][i][:, sl], whole["N_iters"][i][:, sl]))
            for nm in FINALS:
                worst = max(worst, rel_l2(outs[g][nm].cpu().numpy()[:, sl], whole[nm][:, sl]))
        worst_it, worst_fin = _sharded_vs_oracle(ref, world, n, its, outs, cfg.niter)
        print(f"\n[fused peer stores, {world} x, n={n} nt={nt} nfoc={nfoc} regime={regime}] worst deviation from the single context {worst:.1e}; "
              f"each rank's rows against the oracle: per-iteration {worst_it:.2e}, finals {worst_fin:.2e}")
        assert worst <= 1e-6
        assert worst_it <= TOL_ITER and worst_fin <= TOL_FINAL
        # a new batch size drops the attachment loudly instead of exchanging nothing
        mks[0].operand_reserve(nfoc + 1)
        Gd2 = torch.zeros((nfoc + 1, n, nt), dtype=torch.float32, device=dev)
        with pytest.raises(B.MkError):
            mks[0].begin(Gd2, torch.zeros((nfoc + 1, n), dtype=torch.float32, device=dev))
    finally:
        for mk in mks:
            mk.close()


@pytest.mark.parametrize("k,n,nt,nfoc,regime,world", [(1, 37, 512, 3, 1, 2), (3, 150, 2048, 19, 3, 3)])
def test_row_sharded_fused_with_stream_ordered_barriers(k, n, nt, nfoc, regime, world):
    """mk_sync_barrier: the two barriers per synthesis of the fused exchange as stream-ordered flag writes / waits.  Every
    rank runs on a stream of its OWN; the host enqueues the whole run without ever synchronising (one synchronize at the
    very end); the results must equal the single context's bit for bit and meet the oracle."""
    import torch
    from paper_2106_04649_b200 import binding as B, shard
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal="fan:250", niter=5))
    R, Gd, td = problem(cfg)
    whole = gpu_chain(cfg, R, Gd, td, regime=regime)
    ref = _oracle_chain(cfg, R, Gd, td)
    dev = torch.device("cuda:0")
    dR, dGd, dtd = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (R, Gd, td))
    streams = [torch.cuda.Stream(device=dev) for _ in range(world)]
    mks = []
    try:
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            mk = B.Marchenko(n, n, nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(rows.start, len(rows)))
            mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
            mk.set_option(B.MK_OPT_REGIME, regime)
            # every rank ingests ONLY its own receiver rows (mk_load_R_rows), in two uneven shot chunks
            mine = dR[:, rows.start:rows.stop].contiguous()
            cut = max(1, n // 3)
            mk.load_R_rows(mine[:cut], 0)
            mk.load_R_rows(mine[cut:], cut)
            mks.append(mk)
        shard.attach_in_process(mks, nfoc)
        shard.sync_attach_in_process(mks)
        its = [[torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for _ in range(cfg.niter)] for _ in mks]
        outs = [{nm: torch.zeros((nfoc, n, nt), dtype=torch.float32, device=dev) for nm in FINALS} for _ in mks]

        def all_ranks(call):
            for g, mk in enumerate(mks):
                call(g, mk)

        # one lock-step pass on the default stream first, so that every buffer the run needs exists: an allocation in
        # the middle of the real run could make the host wait for a stream that waits for a rank not yet enqueued
        all_ranks(lambda g, mk: mk.begin(dGd, dtd))
        all_ranks(lambda g, mk: mk.operand_exchanged(0))
        all_ranks(lambda g, mk: mk.step_contract())
        all_ranks(lambda g, mk: mk.step_post(None))
        all_ranks(lambda g, mk: mk.operand_exchanged(0))
        for field in (B.MK_FIELD_GMINUS, B.MK_FIELD_GPLUS):
            all_ranks(lambda g, mk: mk.finish_prepare(field))
            all_ranks(lambda g, mk: mk.operand_exchanged(1))
            all_ranks(lambda g, mk: mk.finish_complete(field, outs[g]["G"]))
        torch.cuda.synchronize()                    # inputs, ingest, operands and workspaces are in place
        for g, mk in enumerate(mks):
            mk.set_stream(streams[g].cuda_stream)

        # shard.run_row_sharded_fused, rank by rank in one host thread: only ENQUEUES, the ordering is the streams'
        all_ranks(lambda g, mk: mk.sync_barrier())
        all_ranks(lambda g, mk: mk.begin(dGd, dtd))
        all_ranks(lambda g, mk: mk.sync_barrier())
        all_ranks(lambda g, mk: mk.operand_exchanged(0))
        for i in range(cfg.niter):
            all_ranks(lambda g, mk: mk.step_contract())
            all_ranks(lambda g, mk: mk.sync_barrier())          # every rank has read the operand
            all_ranks(lambda g, mk: mk.step_post(its[g][i]))
            all_ranks(lambda g, mk: mk.sync_barrier())          # every rank's rows have landed everywhere
            all_ranks(lambda g, mk: mk.operand_exchanged(0))
        all_ranks(lambda g, mk: mk.finish({nm: outs[g][nm] for nm in ("f1plus", "f1min", "G")}))
        for name, field in (("Gminus", B.MK_FIELD_GMINUS), ("Gplus", B.MK_FIELD_GPLUS)):
            all_ranks(lambda g, mk: mk.sync_barrier())
            all_ranks(lambda g, mk: mk.finish_prepare(field))
            all_ranks(lambda g, mk: mk.sync_barrier())
            all_ranks(lambda g, mk: mk.operand_exchanged(1))
            all_ranks(lambda g, mk: mk.finish_complete(field, outs[g][name]))
        torch.cuda.synchronize()                    # the only host synchronisation of the run
        worst = 0.0
        np_its = [[t.cpu().numpy() for t in its[g]] for g in range(world)]
        for g in range(world):
            rows = shard.row_slice(n, g, world)
            sl = slice(rows.start, rows.stop)
            for i in range(cfg.niter):
                worst = max(worst, rel_l2(np_its[g][i][:, sl], whole["N_iters"][i][:, sl]))
            for nm in FINALS:
                worst = max(worst, rel_l2(outs[g][nm].cpu().numpy()[:, sl], whole[nm][:, sl]))
        worst_it, worst_fin = _sharded_vs_oracle(ref, world, n, np_its, outs, cfg.niter)
        print(f"\n[stream-ordered barriers, {world} ranks on {world} streams, n={n} nt={nt} nfoc={nfoc} regime={regime}] worst deviation from "
              f"the single context {worst:.1e}; against the oracle: per-iteration {worst_it:.2e}, finals {worst_fin:.2e}")
        assert worst <= 1e-6
        assert worst_it <= TOL_ITER and worst_fin <= TOL_FINAL
    finally:
        torch.cuda.synchronize()
        for mk in mks:
            mk.close()


@pytest.mark.parametrize("nfoc", [1, 2, 4])
def test_fused_finals_match_separate_finals(nfoc):
    """MK_OPT_FUSED_FINALS: with 1, 2 or 4 focal points G^- and G^+ come from ONE pass over R^ (2 nfoc right-hand sides);
    the separate path is the one the chain tests hold against the oracle."""
    cfg = calibrated(configs.scaled(1, n=70, nt=2048 if nfoc == 4 else 512, nfoc=nfoc, focal="single:400" if nfoc == 1 else "fan:250", niter=4))
    R, Gd, td = problem(cfg)
    ref = _oracle_chain(cfg, R, Gd, td)
    import torch
    from paper_2106_04649_b200 import binding as B
    dev = torch.device("cuda:0")
    res = {}
    for fused in (0, 1):
        with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax) as mk:
            mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
            mk.set_option(B.MK_OPT_FUSED_FINALS, fused)
            mk.load_R(torch.from_numpy(R).to(dev))
            outs = {nm: torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in FINALS}
            mk.set_option(B.MK_OPT_TIMING, 1)
            mk.run(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev), cfg.niter, outs)
            torch.cuda.synchronize()
            assert int(mk.get_info(B.MK_INFO_SYN_LAUNCHES)) == cfg.niter + (1 if fused else 2)
            res[fused] = {nm: t.cpu().numpy() for nm, t in outs.items()}
    for nm in FINALS:
        assert rel_l2(res[1][nm], ref[nm]) <= TOL_FINAL, nm
        assert rel_l2(res[1][nm], res[0][nm]) <= 2e-6, nm
