"""NEXT-4: sources and receivers that are not co-located one to one, irregular source spacing —
mk_set_geometry through the whole chain against the oracle's orc_marchenko_geom (pinned in test_oracle_pins.py by the
square scheme on the union grid).  Eq. (1): the integral runs over source positions and is evaluated at
receiver positions; PAPER.md:28 keeps ns and nr apart."""
import numpy as np
import pytest

import oracle
from _util import rel_l2

pytestmark = pytest.mark.gpu

TOL_ITER, TOL_FINAL = 2e-5, 1e-4
FINALS = ("f1plus", "f1min", "G", "Gplus", "Gminus")


def _geometry(ns, nr, seed):
    """Shots and receivers on a common line of positions: every member of the smaller set coincides with a member of the
    larger one, except two that have no partner at all."""
    rng = np.random.default_rng(seed)
    big, small = max(ns, nr), min(ns, nr)
    npos = big + 2
    pos_big = np.sort(rng.choice(npos, big, replace=False))                 # leaves two free positions
    free = np.setdiff1d(np.arange(npos), pos_big)
    pos_small = np.sort(np.concatenate([rng.choice(pos_big, small - 2, replace=False), free]))
    pos_s, pos_r = (pos_big, pos_small) if ns >= nr else (pos_small, pos_big)
    assert len(pos_r) == nr and len(np.unique(pos_r)) == nr
    rec_of_shot = np.array([int(np.nonzero(pos_r == p)[0][0]) if p in pos_r else -1 for p in pos_s], np.int32)
    return pos_s, pos_r, rec_of_shot


@pytest.mark.parametrize("ns,nr,nt,nfoc,regime,custom_w", [
    (48, 37, 256, 3, 1, False),      # more shots than receivers: eleven source positions carry a zero operand
    (37, 48, 256, 3, 1, True),       # more receivers than shots, irregular quadrature weights
    (48, 37, 256, 12, 2, True), (37, 48, 256, 12, 3, False), (150, 133, 128, 40, 3, True),
    (30, 22, 2048, 5, 1, True), (22, 30, 2048, 11, 3, False), (20, 26, 4096, 3, 2, True),   # register-resident transforms
])
def test_non_colocated_spread_matches_the_oracle(ns, nr, nt, nfoc, regime, custom_w):
    import torch
    from paper_2106_04649_b200 import binding as B
    dt, dx, eps, niter = 0.004, 10.0, 3, 6
    fmin, fmax = 10.0, 0.3 / dt
    rng = np.random.default_rng(1000 * ns + nr)
    pos_s, pos_r, rec_of_shot = _geometry(ns, nr, ns + nr)
    assert (rec_of_shot < 0).sum() >= 2 and (rec_of_shot >= 0).sum() >= min(ns, nr) - 2
    w = (rng.uniform(0.5, 1.5, ns) * dx).astype(np.float32) if custom_w else None
    w64 = w.astype(np.float64) if custom_w else oracle.weights(ns, dx)
    R = rng.standard_normal((ns, nr, nt)).astype(np.float32)
    R[:, :, nt // 2:] = 0.0
    Gd = rng.standard_normal((nfoc, nr, nt)).astype(np.float32)
    Gd[:, :, nt // 4:] = 0.0
    td = ((rng.integers(nt // 16, nt // 4, size=(nfoc, nr)) + 0.25) * dt).astype(np.float32)
    o = oracle.marchenko_geom(R, Gd, td, dt, w64, rec_of_shot, fmin, fmax, 2, eps, want=())
    R *= np.float32(2.0 ** np.round(np.log2(0.5 * np.linalg.norm(o["N_iters"][0]) / np.linalg.norm(o["N_iters"][1]))))
    ref = oracle.marchenko_geom(R, Gd, td, dt, w64, rec_of_shot, fmin, fmax, niter, eps)
    dev = torch.device("cuda:0")
    with B.Marchenko(ns, nr, nt, dt, dx, fmin, fmax) as mk:
        mk.set_option(B.MK_OPT_EPS_SAMPLES, eps)
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.set_geometry(rec_of_shot, w)
        cut = max(1, (2 * ns) // 3)
        mk.load_R(torch.from_numpy(R[:cut].copy()).to(dev), 0)
        with pytest.raises(B.MkError) as e:                      # the weights are folded into R^ at ingest
            mk.set_geometry(rec_of_shot, w)
        assert e.value.code == B.MK_ERR_STATE
        mk.load_R(torch.from_numpy(R[cut:].copy()).to(dev), cut)
        mk.begin(torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev))
        buf = torch.empty((nfoc, nr, nt), dtype=torch.float32, device=dev)
        errs = []
        for i in range(niter):
            mk.step(buf)
            errs.append(rel_l2(buf.cpu().numpy(), ref["N_iters"][i]))
        outs = {nm: torch.empty((nfoc, nr, nt), dtype=torch.float32, device=dev) for nm in FINALS}
        mk.finish(outs)
        torch.cuda.synchronize()
        fin = {nm: rel_l2(outs[nm].cpu().numpy(), ref[nm]) for nm in FINALS}
        used = int(mk.get_info(B.MK_INFO_REGIME_USED))
    print(f"\n[ns={ns} nr={nr} nt={nt} nfoc={nfoc} regime={used} weights={'given' if custom_w else 'trapezoid'}] per-iteration max {max(errs):.2e} "
          + " ".join(f"{k}={v:.1e}" for k, v in fin.items()))
    assert np.linalg.norm(ref["N_iters"][-1]) > 1e-6 * np.linalg.norm(ref["N_iters"][0]) > 0
    assert max(errs) <= TOL_ITER, errs
    assert max(fin.values()) <= TOL_FINAL, fin


def test_geometry_argument_checks():
    import torch
    from paper_2106_04649_b200 import binding as B
    with B.Marchenko(6, 4, 64, 0.004, 10.0, 10.0, 100.0) as mk:
        for bad in ([0, 1, 2, 3, 4, 0], [0, 1, 2, 3, 3, -1], [0, 1, 2, 9, -1, -1]):       # wrong range / two shots at one receiver
            with pytest.raises(B.MkError) as e:
                mk.set_geometry(np.array(bad[:6]) if len(bad) == 6 else bad)
            assert e.value.code == B.MK_ERR_INVALID_ARG
        with pytest.raises(B.MkError):
            mk.set_geometry(None, np.array([1, 1, -1, 1, 1, 1], np.float32))
        with pytest.raises(ValueError):
            mk.set_geometry(np.zeros(5, np.int32))
        mk.set_geometry([3, -1, 2, 1, 0, -1], np.full(6, 7.5, np.float32))
        mk.set_geometry(None, None)                                                       # back to the default
    with pytest.raises(B.MkError):                                                        # row sharding: co-located spreads only
        B.Marchenko(6, 4, 64, 0.004, 10.0, 10.0, 100.0, rows=(0, 2))
