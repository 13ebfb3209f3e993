"""Compressed R^ (MK_OPT_RHAT_FORMAT = 1, "q16": block floating point with int16 mantissas, one fp32 scale per 16 shots;
SURVEY.md section 8(f) NEXT-4) for the bandwidth-bound regime.  Two questions, two references:

 (a) is the ARITHMETIC right?  The format is restated here in numpy (q16_model: the definition in include/mk.h written
     out), applied to the spectrum of R, and the de-quantised response is handed to the fp64 oracle as its R.  Against
     that reference the CUDA path must be as good as the uncompressed one, up to the few mantissas whose rounding falls
     the other way because the GPU quantises an fp32 FFT and numpy an fp64 one (a flip changes one component by one
     step; about 0.3 % of the components flip, which is ~0.2 of the quantisation error itself).
 (b) what does the compression COST?  Against the oracle on the uncompressed R the path is held to its own stated
     tolerance: relative L2 <= 5e-4 per iteration and <= 1e-3 on the final fields.  north_star's
     2e-5 / 1e-4 cannot hold for a lossy format and is not claimed.
"""
import numpy as np
import pytest

import oracle
from paper_2106_04649_b200 import configs
from _util import calibrated, gpu_chain, problem, rel_l2

pytestmark = pytest.mark.gpu

TOL_Q_ITER, TOL_Q_FINAL = 5e-4, 1e-3
FINALS = ("f1plus", "f1min", "G", "Gplus", "Gminus")


def q16_model(R, dt, dx, fmin, fmax):
    """R [shot][rec][nt] fp32 -> the time-domain response whose band-limited spectrum is the q16 representation of R's.
    Per (receiver, bin) row, blocks of 16 shots: sc = max(|re|, |im|) / 32767, q = rint(v / sc), value = q * sc."""
    ns, nr, nt = R.shape
    w = oracle.weights(ns, dx)
    klo, khi, nb = oracle.band(nt, dt, fmin, fmax)
    spec = np.fft.rfft(R.astype(np.float64), axis=-1)[:, :, klo:khi + 1] * (dt * w)[:, None, None]
    ld = -(-ns // 16) * 16
    v = np.zeros((ld, nr, nb, 2), np.float32)
    v[:ns, :, :, 0] = spec.real
    v[:ns, :, :, 1] = spec.imag
    blk = v.reshape(ld // 16, 16, nr, nb, 2)
    m = np.abs(blk).max(axis=(1, 4), keepdims=True).astype(np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = np.where(m > 0, np.float32(32767) / m, np.float32(0)).astype(np.float32)
    q = np.clip(np.rint(blk * inv), -32767, 32767).astype(np.float32)
    deq = (q * (m / np.float32(32767))).reshape(ld, nr, nb, 2)[:ns].astype(np.float64)
    full = np.zeros((ns, nr, nt // 2 + 1), np.complex128)
    full[:, :, klo:khi + 1] = (deq[..., 0] + 1j * deq[..., 1]) / (dt * w)[:, None, None]
    return np.fft.irfft(full, n=nt, axis=-1).astype(np.float32)


@pytest.mark.parametrize("k,n,nt,nfoc", [(1, 70, 512, 1), (1, 70, 512, 4), (1, 45, 2048, 1), (3, 90, 512, 7), (4, 40, 1024, 8)])
def test_q16_chain_against_both_references(k, n, nt, nfoc):
    focal = "single:400" if nfoc == 1 else "fan:250"
    cfg = calibrated(configs.scaled(k, n=n, nt=nt, nfoc=nfoc, focal=focal, niter=8))
    R, Gd, td = problem(cfg)
    got = gpu_chain(cfg, R, Gd, td, rhat_format=1)
    assert got["regime_used"] == 1
    run = lambda RR: oracle.marchenko(RR, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, cfg.niter, cfg.eps)
    ref, ref_q = run(R), run(q16_model(R, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax))
    cost = [rel_l2(got["N_iters"][i], ref["N_iters"][i]) for i in range(cfg.niter)]
    arith = [rel_l2(got["N_iters"][i], ref_q["N_iters"][i]) for i in range(cfg.niter)]
    fcost = {nm: rel_l2(got[nm], ref[nm]) for nm in FINALS}
    farith = {nm: rel_l2(got[nm], ref_q[nm]) for nm in FINALS}
    fmt = {nm: rel_l2(ref_q[nm], ref[nm]) for nm in FINALS}
    print(f"\n[q16 {cfg.name} n={n} nt={nt} nfoc={nfoc}] cost of the format: per-iter max {max(cost):.2e}, finals max {max(fcost.values()):.2e} "
          f"(oracle on de-quantised R vs oracle: {max(fmt.values()):.2e}); arithmetic: per-iter max {max(arith):.2e}, finals max {max(farith.values()):.2e}")
    assert max(cost) <= TOL_Q_ITER, cost
    assert max(fcost.values()) <= TOL_Q_FINAL, fcost
    # (a): against the format-aware reference the error is rounding flips (a fraction of the format's own error) + fp32
    assert max(arith) <= 2e-5 + 0.4 * max(cost), (arith, cost)
    assert max(farith.values()) <= 2e-5 + 0.4 * max(fcost.values()), (farith, fcost)


def test_q16_state_and_argument_rules():
    import torch
    from paper_2106_04649_b200 import binding as B
    n, nt = 40, 256
    dev = torch.device("cuda:0")
    R = torch.zeros((n, n, nt), device=dev)
    with B.Marchenko(n, n, nt, 0.004, 10.0, 5.0, 60.0) as mk:
        mk.set_option(B.MK_OPT_RHAT_FORMAT, 1)
        assert mk.get_info(B.MK_INFO_RHAT_BYTES_STORED) == 4.25 * n * mk.get_info(B.MK_INFO_NB) * mk.get_info(B.MK_INFO_LD_SHOT)
        with pytest.raises(B.MkError) as e:
            mk.load_R(R[:10], 0)                     # not a whole number of 16-shot blocks
        assert e.value.code == B.MK_ERR_INVALID_ARG
        mk.load_R(R[:32], 0)
        mk.load_R(R[32:], 32)                        # the ragged tail at the last shot is fine
        with pytest.raises(B.MkError) as e:
            mk.set_option(B.MK_OPT_RHAT_FORMAT, 0)   # R^ is converted at ingest
        assert e.value.code == B.MK_ERR_STATE
        Gd = torch.zeros((9, n, nt), device=dev)
        td = torch.full((9, n), 0.1, device=dev)
        with pytest.raises(B.MkError) as e:
            mk.begin(Gd, td)                         # nine focal points leave the streaming regime
        assert e.value.code == B.MK_ERR_INVALID_ARG
        mk.begin(Gd[:8], td[:8])
    with B.Marchenko(n, n, nt, 0.004, 10.0, 5.0, 60.0, streamed=(10, 5)) as mk:
        with pytest.raises(B.MkError) as e:
            mk.set_option(B.MK_OPT_RHAT_FORMAT, 1)
        assert e.value.code == B.MK_ERR_STATE
