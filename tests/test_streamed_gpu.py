"""Out-of-core R^ (mk_create_streamed, second half): most rows of
R^ live in pinned host memory and pass through two windows in HBM during every contraction.  Row blocks are independent,
so the streamed context must reproduce the resident one BIT FOR BIT in every regime — and, like it, meet the fp64 oracle
to the north_star tolerances.  Also checked: the bytes the contractions report as copied (the passes alternate direction
and reuse the two blocks left in the windows), a reload of R between runs, and the degenerate window shapes."""
import numpy as np
import pytest

import oracle
from paper_2106_04649_b200 import configs
from _util import calibrated, gpu_chain, problem, rel_l2

pytestmark = pytest.mark.gpu

TOL_ITER, TOL_FINAL = 2e-5, 1e-4
FINALS = ("f1plus", "f1min", "G", "Gplus", "Gminus")


def _oracle_chain(cfg, R, Gd, td):
    return oracle.marchenko(R, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, cfg.niter, cfg.eps)


@pytest.mark.parametrize("k,n,nt,nfoc,regime,resident,window", [
    (1, 70, 512, 1, 1, 17, 12),      # 53 host rows in blocks of 12, 12, 12, 12, 5 (ragged tail), streaming GEMV
    (1, 70, 512, 4, 1, 0, 9),        # nothing resident; fused finals (8 right-hand sides)
    (3, 90, 512, 19, 2, 22, 16),     # FFMA GEMM: blocks smaller than its 128-row tile
    (3, 300, 2048, 19, 3, 75, 100),  # tcgen05 GEMM: one TMA descriptor per window, blocks of 100, 100, 25 rows
    (2, 70, 512, 70, 3, 30, 40),     # a single window holds every host row: transferred once, reused ever after
])
def test_streamed_context_reproduces_the_resident_one(k, n, nt, nfoc, regime, resident, window):
    focal = "single:400" if nfoc == 1 else ("line:300" if nfoc == n else "fan:250")
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal=focal, niter=6))
    R, Gd, td = problem(cfg)
    whole = gpu_chain(cfg, R, Gd, td, regime=regime)
    part = gpu_chain(cfg, R, Gd, td, regime=regime, streamed=(resident, window))
    assert part["regime_used"] == whole["regime_used"] == regime
    for nm in FINALS + ("N_iters",):
        assert np.array_equal(part[nm], whole[nm]), f"{nm}: streamed and resident contexts differ"
    ref = _oracle_chain(cfg, R, Gd, td)
    errs = [rel_l2(part["N_iters"][i], ref["N_iters"][i]) for i in range(cfg.niter)]
    ferr = {nm: rel_l2(part[nm], ref[nm]) for nm in FINALS}
    print(f"\n[streamed {cfg.name} n={n} nfoc={nfoc} regime={regime} resident {resident} window {window}] per-iter max {max(errs):.2e} "
          + " ".join(f"{a}={b:.1e}" for a, b in ferr.items()))
    assert max(errs) <= TOL_ITER, errs
    assert max(ferr.values()) <= TOL_FINAL, ferr
    # transfer accounting: the first pass brings every host row in, every later pass all but the two blocks (one, when
    # there is a single window) that the pass before left behind
    row_bytes = whole["rhat_bytes_padded"] / n
    nhost = n - resident
    B = -(-nhost // window)
    rows_of = [min(window, nhost - b * window) for b in range(B)]
    fused = regime == 1 and nfoc in (1, 2, 4)
    passes = cfg.niter + (1 if fused else 2)
    expect, held, rev = 0, set(), False
    for _ in range(passes):
        order = list(range(B))[::-1] if rev else list(range(B))
        for b in order:
            if b not in held:
                expect += rows_of[b]
            held = {x for x in held if (x & 1) != (b & 1)} | {b}
        rev = not rev
    assert part["h2d_bytes"] == pytest.approx(expect * row_bytes), (part["h2d_bytes"] / row_bytes, expect)
    assert whole["h2d_bytes"] == 0


def test_streamed_synthesis_and_reload():
    """mk_synthesis on a streamed context; replacing shots afterwards invalidates what the windows hold."""
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt, nfoc = 40, 256, 3
    rng = np.random.default_rng(5)
    R = rng.standard_normal((n, n, nt)).astype(np.float32)
    R[:, :, nt // 2:] = 0
    R2 = R.copy()
    R2[10:20] = rng.standard_normal((10, n, nt)).astype(np.float32)
    R2[10:20, :, nt // 2:] = 0
    N = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    dt, dx, fmin, fmax = 0.004, 10.0, 5.0, 60.0
    dev = torch.device("cuda:0")
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, fmin, fmax)
    with B.Marchenko(n, n, nt, dt, dx, fmin, fmax, streamed=(8, 5)) as mk:
        assert mk.get_info(B.MK_INFO_RESIDENT_ROWS) == 8 and mk.get_info(B.MK_INFO_WINDOW_ROWS) == 5
        mk.load_R(torch.from_numpy(R).to(dev))
        dN = torch.from_numpy(N).to(dev)
        dS = torch.empty_like(dN)
        for _ in range(2):   # the second pass walks the blocks backwards
            mk.synthesis(dN, dS)
            assert rel_l2(dS.cpu().numpy(), oracle.synthesis(R, N, dt, w, klo, khi)) <= TOL_ITER
        mk.load_R(torch.from_numpy(R2[10:20].copy()).to(dev), 10)
        mk.synthesis(dN, dS)
        assert rel_l2(dS.cpu().numpy(), oracle.synthesis(R2, N, dt, w, klo, khi)) <= TOL_ITER
